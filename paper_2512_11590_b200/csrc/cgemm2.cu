// cgemm2.cu -- PERSISTENT planar complex64 GEMM on tcgen05 (kind::tf32): the trailing update A22 -= L21 U12 of the
// low-precision LU (Eq. 5) and the products of its blocked triangular solves.
//
//   C <- beta*C + alpha*A*B,   A m x k, B k x n, C m x n, each a pair of column-major float planes (re, im).
//
// Same arithmetic and operand layouts as cgemm.cu (four real UMMAs per k-step on the planes as they lie in memory: "4M",
// 8 real flops per complex multiply-add = the 8N^3/3 convention of PAPER.md:190), different execution structure:
//   * persistent: one CTA (NCTA = 1) or one CTA PAIR (NCTA = 2, a cluster of two CTAs on the two SMs of a TPC) per SM
//     walks a static, rasterised sequence of output tiles -- tiles in flight form a compact block of C and move through K
//     nearly in lock step, so every A / B slice is fetched from HBM about once;
//   * the accumulators (Dr | Di, 2 x 128 TMEM columns) are DOUBLE BUFFERED: the epilogue of tile t (tcgen05.ld ->
//     beta*C + alpha*acc -> global) overlaps the main loop of tile t + 1;
//   * NCTA = 2: tcgen05.mma.cta_group::2 with M = 256: each CTA stages its own 128 rows of A and HALF of the B columns, so a
//     k-step reads 6 KB instead of 8 KB of shared memory per CTA (the 128 x 128 single-CTA tile sits exactly at the
//     shared-memory operand bandwidth of the tensor core); only the leader CTA issues MMAs, completion is multicast to
//     both CTAs' barriers.
// Roles per CTA (10 warps): warp 0 TMA producer (one lane), warp 1 TMEM allocator + MMA issuer (one lane, leader CTA only),
// warps 2-9 epilogue (two per TMEM lane quarter 32*(warp%4), half of the tile's columns each).
// Optional in the epilogue: count the results with |re| + |im| > thr (the multiplier check of the block panel, toplu.cu).
#include "lu.cuh"
#include "sm100.cuh"

namespace hp {

// SMs a persistent launch leaves free (look-ahead: the deferred update runs beside the next panel's chain of small kernels,
// which need an SM with free shared memory and TMEM to start at all).  Host-thread-local, set for the duration of the enqueue.
static thread_local int g_sm_reserve = 0;
int sm_reserve_in_force() { return g_sm_reserve; }
ScopedSmReserve::ScopedSmReserve(int sms) : prev(g_sm_reserve) { g_sm_reserve = sms; }
ScopedSmReserve::~ScopedSmReserve() { g_sm_reserve = prev; }

using namespace sm100;

int make_map(CUtensorMap *map, const float *plane, long rows, long cols, long ld, int box_rows, int box_cols,
             CUtensorMapSwizzle swz);  // cgemm.cu

namespace {

constexpr int G2_BM = 128;   // rows of C per CTA (UMMA M = 128 * NCTA)
constexpr int G2_KC = 32;    // floats of K per stage = one 128-byte swizzle row
constexpr int G2_EPI = 8;                 // epilogue warps: two per TMEM lane quarter, each takes half of the tile's columns
constexpr int G2_NT = 64 + 32 * G2_EPI;   // (the epilogue's global loads are latency-bound: bytes in flight scale with its warps)
constexpr int G2_MAX_WAVES = 256;  // counters of the wave barrier (G2Args::wave_ctr)
constexpr int G2_TMEM = 512; // BN = 128: two accumulator stages of (Dr | Di) = 2 x 2 x 128 columns; BN = 256: one stage

template <int NCTA, int BN> struct G2Cfg {
    static constexpr int ACC = G2_TMEM / (2 * BN);                   // accumulator stages
    static constexpr int BNL = BN / NCTA;                            // B columns staged by one CTA
    static constexpr int A_PLANE = G2_BM * G2_KC * 4;                // 16 KB
    static constexpr int B_PLANE = BNL * G2_KC * 4;                  // 16 KB / 8 KB
    static constexpr int STAGE = 2 * A_PLANE + 2 * B_PLANE;          // 64 KB / 48 KB
    static constexpr int STAGES = (200 * 1024) / STAGE;              // 3 (64 KB stages) or 4 (48 KB)
    static constexpr int SMEM = STAGES * STAGE + 1024 /* alignment slack */ + 256 /* barriers */;
};

struct G2Maps {
    CUtensorMap a_re, a_im, b_re, b_im;
};

struct G2Args {
    int M, N, K;
    float alpha, beta;
    float *Cre, *Cim;
    long ldc;
    int tiles_m, tiles_n;   // tiles_m counts (128 * NCTA)-row tiles
    int group;              // rasterisation group (tile rows walked before stepping a tile column)
    float chk_thr;          // epilogue check: count |re| + |im| > chk_thr (or NaN) into *chk_count when non-null
    int *chk_count;
    unsigned *wave_ctr;     // non-null: one zeroed counter per wave of tiles; the producers of all CTAs meet before each wave
};

template <int NCTA, int BN>
__global__ void __launch_bounds__(G2_NT, 1)
    cgemm2_kernel(const __grid_constant__ G2Maps maps, const G2Args p) {
    typedef G2Cfg<NCTA, BN> Cfg;
    constexpr int G2_BN = BN;
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + Cfg::STAGES * Cfg::STAGE);
    uint64_t *empty = full + Cfg::STAGES;
    uint64_t *tmem_full = empty + Cfg::STAGES;   // [2]
    uint64_t *tmem_empty = tmem_full + 2;        // [2]
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tmem_empty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = NCTA == 2 ? cluster_ctarank() : 0u;
    const bool leader = rank == 0;
    const int cluster_id = (int)blockIdx.x / NCTA, nclusters = (int)gridDim.x / NCTA;
    const int ntiles = p.tiles_m * p.tiles_n;
    const int nk = (p.K + G2_KC - 1) / G2_KC;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&maps.a_re);
        tma_prefetch_desc(&maps.a_im);
        tma_prefetch_desc(&maps.b_re);
        tma_prefetch_desc(&maps.b_im);
        for (int s = 0; s < Cfg::STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 1);
        }
        for (int a = 0; a < Cfg::ACC; ++a) {
            mbar_init(&tmem_full[a], 1);
            mbar_init(&tmem_empty[a], G2_EPI * NCTA);  // one arrival per epilogue warp of every CTA of the pair
        }
        fence_mbar_init();
    }
    if (warp == 1) {
        if constexpr (NCTA == 2) tmem_alloc_pair<G2_TMEM>(tmem_slot);
        else tmem_alloc<G2_TMEM>(tmem_slot);
    }
    tc_fence_before();
    __syncthreads();
    if constexpr (NCTA == 2) cluster_sync_all();  // the peer's barriers are initialised before anything arrives on them
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    pdl_wait();     // the prologue above may overlap the predecessor's tail (launch_pdl); global memory only from here on
    pdl_trigger();

    if (warp == 0) {
        // ================================================================================ TMA producer
        if (lane == 0) {
            const uint32_t full0 = NCTA == 2 ? mapa_u32(smem_u32(&full[0]), 0) : smem_u32(&full[0]);
            long it = 0;
            int wave = 0;
            for (int t = cluster_id; t < ntiles; t += nclusters, ++wave) {
                if (p.wave_ctr != nullptr && wave > 0) {
                    // Wave barrier: CTA pairs that finish a tile early would otherwise run ahead into the next wave alone and
                    // stream its operands from HBM a second time when the others follow (L2 holds ~100 k-steps of a wave).
                    // Alone on the GPU all CTAs that own a tile in this wave are resident (one CTA per SM, grid <= SM count); it
                    // costs one L2 round trip per tile of >= 100 us.
                    const unsigned parts = (unsigned)min(nclusters, ntiles - wave * nclusters) * NCTA;
                    // The barrier is a traffic optimisation, not a correctness requirement, and it must not be able to hang: when
                    // another stream's kernels hold SMs (several contexts, look-ahead), part of this grid may not be resident
                    // yet -- so the wait is bounded (~150 us) and then simply gives up.
                    atomicAdd(&p.wave_ctr[wave], 1u);
                    const long long t_give_up = clock64() + 300000;
                    while (*(volatile unsigned *)&p.wave_ctr[wave] < parts && clock64() < t_give_up) {
                    }
                }
                int tm, tn;
                raster(t, p.tiles_m, p.tiles_n, p.group, tm, tn);
                const int m0 = tm * (G2_BM * NCTA) + (int)rank * G2_BM;
                const int n0 = tn * G2_BN + (int)rank * Cfg::BNL;
                for (int kt = 0; kt < nk; ++kt, ++it) {
                    const int s = (int)(it % Cfg::STAGES);
                    const uint32_t ph = (uint32_t)(it / Cfg::STAGES) & 1;
                    mbar_wait(&empty[s], ph ^ 1);
                    if (leader) mbar_expect_tx(&full[s], Cfg::STAGE * NCTA);  // both CTAs' halves land on the leader's barrier
                    unsigned char *st = smem + s * Cfg::STAGE;
                    const uint32_t bar = full0 + (uint32_t)(s * sizeof(uint64_t));
                    const int k0 = kt * G2_KC;
#pragma unroll
                    for (int c = 0; c < G2_BM / 32; ++c) {
                        if constexpr (NCTA == 2) {
                            tma_load_2d_pair(st + c * (G2_KC * 128), &maps.a_re, bar, m0 + 32 * c, k0);
                            tma_load_2d_pair(st + Cfg::A_PLANE + c * (G2_KC * 128), &maps.a_im, bar, m0 + 32 * c, k0);
                        } else {
                            tma_load_2d(st + c * (G2_KC * 128), &maps.a_re, &full[s], m0 + 32 * c, k0);
                            tma_load_2d(st + Cfg::A_PLANE + c * (G2_KC * 128), &maps.a_im, &full[s], m0 + 32 * c, k0);
                        }
                    }
                    if constexpr (NCTA == 2) {
                        tma_load_2d_pair(st + 2 * Cfg::A_PLANE, &maps.b_re, bar, k0, n0);
                        tma_load_2d_pair(st + 2 * Cfg::A_PLANE + Cfg::B_PLANE, &maps.b_im, bar, k0, n0);
                    } else {
                        tma_load_2d(st + 2 * Cfg::A_PLANE, &maps.b_re, &full[s], k0, n0);
                        tma_load_2d(st + 2 * Cfg::A_PLANE + Cfg::B_PLANE, &maps.b_im, &full[s], k0, n0);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ================================================================================ MMA issuer (leader CTA only)
        if (lane == 0 && leader) {
            constexpr uint32_t ID = idesc_tf32(G2_BM * NCTA, G2_BN, 1, 0, 0, 0);
            constexpr uint32_t ID_NEGA = idesc_tf32(G2_BM * NCTA, G2_BN, 1, 0, 1, 0);
            long it = 0;
            int ti = 0;
            for (int t = cluster_id; t < ntiles; t += nclusters, ++ti) {
                const int a = ti % Cfg::ACC;
                const uint32_t aph = (uint32_t)(ti / Cfg::ACC) & 1;
                mbar_wait(&tmem_empty[a], aph ^ 1);  // the epilogues of tile ti - ACC have drained this accumulator stage
                tc_fence_after();
                const uint32_t d_re = tmem + (uint32_t)(a * 2 * G2_BN), d_im = d_re + G2_BN;
                for (int kt = 0; kt < nk; ++kt, ++it) {
                    const int s = (int)(it % Cfg::STAGES);
                    const uint32_t ph = (uint32_t)(it / Cfg::STAGES) & 1;
                    mbar_wait(&full[s], ph);
                    tc_fence_after();
                    const uint32_t a_re = smem_u32(smem + s * Cfg::STAGE), a_im = a_re + Cfg::A_PLANE;
                    const uint32_t b_re = a_re + 2 * Cfg::A_PLANE, b_im = b_re + Cfg::B_PLANE;
#pragma unroll
                    for (int ks = 0; ks < G2_KC / 8; ++ks) {
                        const uint64_t dar = smem_desc_sw128_base32(a_re + ks * 1024, G2_KC * 128, 512);
                        const uint64_t dai = smem_desc_sw128_base32(a_im + ks * 1024, G2_KC * 128, 512);
                        const uint64_t dbr = smem_desc_sw128(b_re + ks * 32, 16, 1024);
                        const uint64_t dbi = smem_desc_sw128(b_im + ks * 32, 16, 1024);
                        const uint32_t acc = (kt | ks) ? 1u : 0u;
                        if constexpr (NCTA == 2) {
                            umma_tf32_pair(d_re, dar, dbr, ID, acc);  // alternate the accumulators: no back-to-back
                            umma_tf32_pair(d_im, dar, dbi, ID, acc);  // dependent MMAs
                            umma_tf32_pair(d_re, dai, dbi, ID_NEGA, 1u);
                            umma_tf32_pair(d_im, dai, dbr, ID, 1u);
                        } else {
                            umma_tf32(d_re, dar, dbr, ID, acc);
                            umma_tf32(d_im, dar, dbi, ID, acc);
                            umma_tf32(d_re, dai, dbi, ID_NEGA, 1u);
                            umma_tf32(d_im, dai, dbr, ID, 1u);
                        }
                    }
                    if constexpr (NCTA == 2) umma_commit_pair(&empty[s]);
                    else umma_commit(&empty[s]);
                }
                if constexpr (NCTA == 2) umma_commit_pair(&tmem_full[a]);
                else umma_commit(&tmem_full[a]);
            }
        }
    } else {
        // ================================================================================ epilogue
        const int q = warp & 3;  // TMEM lane quarter this warp may access
        constexpr int EC = G2_BN / (G2_EPI / 4);       // columns per epilogue warp
        const int cbeg = ((warp - 2) >> 2) * EC;       // first column of this warp's share
        const uint32_t te0 = NCTA == 2 ? mapa_u32(smem_u32(&tmem_empty[0]), 0) : smem_u32(&tmem_empty[0]);
        int bad = 0;
        int ti = 0;
        for (int t = cluster_id; t < ntiles; t += nclusters, ++ti) {
            const int a = ti % Cfg::ACC;
            const uint32_t aph = (uint32_t)(ti / Cfg::ACC) & 1;
            int tm, tn;
            raster(t, p.tiles_m, p.tiles_n, p.group, tm, tn);
            const int n0 = tn * G2_BN;
            const long row = (long)tm * (G2_BM * NCTA) + (long)rank * G2_BM + 32 * q + lane;
            const bool row_ok = row < p.M;
            mbar_wait(&tmem_full[a], aph);
            tc_fence_after();
            const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16) + (uint32_t)(a * 2 * G2_BN);
            // the old C values of chunk i + 1 are requested before chunk i is stored: twice the loads in flight per warp
            float oldr[2][16], oldi[2][16];
            auto load_old = [&](int c0, float (&orr)[16], float (&oii)[16]) {
                if (p.beta == 0.f) return;
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const long col = (long)n0 + c0 + j;
                    const bool ok = row_ok && col < p.N;
                    orr[j] = ok ? p.Cre[col * p.ldc + row] : 0.f;
                    oii[j] = ok ? p.Cim[col * p.ldc + row] : 0.f;
                }
            };
            load_old(cbeg, oldr[0], oldi[0]);
#pragma unroll
            for (int ci = 0; ci < EC / 16; ++ci) {
                const int c0 = cbeg + 16 * ci;
                if (n0 + c0 >= p.N) break;  // warp-uniform
                uint32_t ar[16], ai[16];
                if (nk > 0) {
                    tmem_ld16(lane_base + c0, ar);
                    tmem_ld16(lane_base + G2_BN + c0, ai);
                }
                if (ci + 1 < EC / 16) load_old(c0 + 16, oldr[(ci + 1) & 1], oldi[(ci + 1) & 1]);
                if (nk > 0) {
                    tmem_ld_wait();
                } else {
#pragma unroll
                    for (int j = 0; j < 16; ++j) ar[j] = ai[j] = 0u;
                }
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const long col = (long)n0 + c0 + j;
                    if (row_ok && col < p.N) {
                        float vr = p.alpha * __uint_as_float(ar[j]), vi = p.alpha * __uint_as_float(ai[j]);
                        if (p.beta != 0.f) {
                            vr = fmaf(p.beta, oldr[ci & 1][j], vr);
                            vi = fmaf(p.beta, oldi[ci & 1][j], vi);
                        }
                        p.Cre[col * p.ldc + row] = vr;
                        p.Cim[col * p.ldc + row] = vi;
                        if (p.chk_count != nullptr && !(fabsf(vr) + fabsf(vi) <= p.chk_thr)) bad = 1;
                    }
                }
            }
            // this warp has read its quarter of the accumulator stage: hand it back to the MMA issuer (leader CTA)
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                if constexpr (NCTA == 2) mbar_arrive_cluster(te0 + (uint32_t)(a * sizeof(uint64_t)));
                else mbar_arrive(&tmem_empty[a]);
            }
        }
        if (p.chk_count != nullptr && __any_sync(0xffffffffu, bad) && lane == 0) atomicAdd(p.chk_count, 1);
    }
    tc_fence_before();
    __syncthreads();
    if constexpr (NCTA == 2) cluster_sync_all();  // the leader's MMAs read the peer's shared memory and write its TMEM
    if (warp == 1) {
        if constexpr (NCTA == 2) tmem_dealloc_pair<G2_TMEM>(tmem);
        else tmem_dealloc<G2_TMEM>(tmem);
    }
}

template <int NCTA, int BN>
int launch_cgemm2(cudaStream_t st, int m, int n, int k, float alpha, CView A, CView B, float beta, CView C, float chk_thr,
                  int *chk_count, unsigned *wave_ctr) {
    typedef G2Cfg<NCTA, BN> Cfg;
    constexpr int G2_BN = BN;
    auto kern = cgemm2_kernel<NCTA, BN>;
    static SmemCfg cfg;
    HP_TRY(configure_smem(cfg, kern, Cfg::SMEM));
    G2Maps maps;
    const int kk = k > 0 ? k : 1;
    HP_TRY(make_map(&maps.a_re, A.re, m, kk, A.ld, 32, G2_KC, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B));
    HP_TRY(make_map(&maps.a_im, A.im, m, kk, A.ld, 32, G2_KC, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B));
    HP_TRY(make_map(&maps.b_re, B.re, kk, n, B.ld, G2_KC, Cfg::BNL, CU_TENSOR_MAP_SWIZZLE_128B));
    HP_TRY(make_map(&maps.b_im, B.im, kk, n, B.ld, G2_KC, Cfg::BNL, CU_TENSOR_MAP_SWIZZLE_128B));
    G2Args p;
    p.M = m; p.N = n; p.K = k;
    p.alpha = alpha; p.beta = beta;
    p.Cre = C.re; p.Cim = C.im; p.ldc = C.ld;
    p.tiles_m = ceil_div(m, G2_BM * NCTA);
    p.tiles_n = ceil_div(n, G2_BN);
    // tiles in flight (74 pair tiles of 256 x BN, or 148 of 128 x 128) cover a square-ish block of C
    p.group = NCTA == 2 ? (BN == 256 ? 8 : 6) : 12;
    p.chk_thr = chk_thr;
    p.chk_count = chk_count;
    const long ntiles = (long)p.tiles_m * p.tiles_n;
    const int nclusters = (int)std::min<long>(ntiles, (kNumSMs - sm_reserve_in_force()) / NCTA);
    const long waves = (ntiles + nclusters - 1) / nclusters;
    p.wave_ctr = nullptr;
    if (wave_ctr != nullptr && waves > 1 && waves <= G2_MAX_WAVES && k >= 1024) {  // long tiles only: the barrier is per tile
        HP_CUDA(cudaMemsetAsync(wave_ctr, 0, sizeof(unsigned) * (size_t)waves, st));
        p.wave_ctr = wave_ctr;
    }
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3(nclusters * NCTA);
    lc.blockDim = dim3(G2_NT);
    lc.dynamicSmemBytes = Cfg::SMEM;
    lc.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = NCTA;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    lc.attrs = attr;
    lc.numAttrs = (pdl_enabled() && p.wave_ctr == nullptr) ? 2 : 1;  // behind the counters' memset: a plain dependency
    HP_CUDA(cudaLaunchKernelEx(&lc, kern, maps, p));
    HP_LAUNCHED();
    return 0;
}

}  // namespace

// C <- beta*C + alpha*A*B on split-complex float planes, persistent kernel.  shape: 0 = single CTAs, 128 x 128 tiles;
// 1 = CTA pairs, 256 x 128 tiles (double-buffered accumulators); 2 = CTA pairs, 256 x 256 tiles (all of TMEM is one stage).
// Same argument rules as cgemm (cgemm.cu).  C may alias B when m <= 128 and beta == 0 (pair == false), and A when
// n <= 128 and beta == 0.  chk_count != nullptr: *chk_count is incremented (by some positive amount) if any result has
// |re| + |im| > chk_thr or is NaN.
int cgemm2(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C, int shape, float chk_thr,
           int *chk_count, unsigned *wave_ctr) {
    if (m <= 0 || n <= 0) return 0;
    if (k <= 0 && beta == 1.0 && !chk_count) return 0;
    if (((uintptr_t)A.re | (uintptr_t)A.im | (uintptr_t)B.re | (uintptr_t)B.im) & 15) return -6;
    if ((A.ld | B.ld) & 3) return -7;
    if (shape == 2) return launch_cgemm2<2, 256>(st, m, n, k, (float)alpha, A, B, (float)beta, C, chk_thr, chk_count, wave_ctr);
    if (shape == 1) return launch_cgemm2<2, 128>(st, m, n, k, (float)alpha, A, B, (float)beta, C, chk_thr, chk_count, wave_ctr);
    return launch_cgemm2<1, 128>(st, m, n, k, (float)alpha, A, B, (float)beta, C, chk_thr, chk_count, wave_ctr);
}

}  // namespace hp
