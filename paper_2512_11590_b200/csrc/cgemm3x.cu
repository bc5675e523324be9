// cgemm3x.cu -- planar complex64 GEMM with FP32-CLASS accuracy on the 5th-generation tensor cores ("3xTF32" on tcgen05):
// the products of the complex64 LU when its matrix is too ill-conditioned for single-pass TF32 -- the literal Type-3 Schur
// matrix (kappa ~ 1e5) and the raw mixed solve beyond kappa ~ 1e3 (the paper's
// single-precision factors work while kappa u_FP32 < 1).
//
//   C <- beta*C + alpha*A*B,  operands and layouts as cgemm.cu.
//
// Every FP32 operand x is split as x = hi + lo and every real product is three UMMAs: hi*hi + hi*lo + lo*hi.  The tensor core
// reads its operands from shared memory and uses only the upper 19 bits of an FP32 word (kind::tf32 TRUNCATES), so
//   hi = the word TMA landed, as it is (the hardware sees trunc(x)),
//   lo = rne_tf32(x - trunc(x))  (x - trunc(x) is exact in FP32 and < 2^-10 |x|; rounded to 10 mantissa bits here so that the
//        hardware's truncation of lo is exact),
// which leaves the dropped lo*lo term and the rounding of lo: <= 2^-21 relative.  Four "splitter" warps compute lo from the
// landed tile into a second tile of the same swizzled layout (the transform is elementwise), fence the async proxy and hand
// the stage to the MMA issuer.  The accuracy test (tests/test_gpu_mixed.py, 2^-20 bound) fails if the hardware did anything
// but truncate.
//
// CTA = 10 warps: warp 0 TMA producer, warp 1 TMEM allocator + UMMA issuer, warps 2-5 epilogue, warps 6-9 splitters.
// PERSISTENT: one CTA per SM walks the rasterised tile sequence; two accumulator stages in TMEM, so the epilogue of a tile
// overlaps the main loop of the next.  Tile 128 x 128, K step 16, three stages of (A, B, A_lo, B_lo) = 3 x 64 KB.  (N = 128 halves the shared-memory reads per
// flop of the 128 x 64 version, which was bound by them: 150 -> see DESIGN.md section 8.)
#include <atomic>

#include "lu.cuh"
#include "sm100.cuh"

namespace hp {

using namespace sm100;

int make_map(CUtensorMap *map, const float *plane, long rows, long cols, long ld, int box_rows, int box_cols,
             CUtensorMapSwizzle swz);  // cgemm.cu

namespace {

constexpr int X3_BM = 128, X3_BN = 128, X3_KC = 16, X3_NT = 320;
constexpr int X3_A_PLANE = X3_BM * X3_KC * 4;                 // 8 KB
constexpr int X3_B_PLANE = X3_BN * X3_KC * 4;                 // 8 KB
constexpr int X3_HALF = 2 * X3_A_PLANE + 2 * X3_B_PLANE;      // 32 KB: the TMA-written tiles of one stage
constexpr int X3_STAGE = 2 * X3_HALF;                         // + the lo tiles
constexpr int X3_STAGES = 3;
constexpr int X3_SMEM = X3_STAGES * X3_STAGE + 1024 + 256;
constexpr int X3_ACC = 2;                                     // accumulator stages (Dr | Di each) in TMEM
constexpr int X3_TMEM = X3_ACC * 2 * X3_BN;                   // all 512 columns

struct X3Maps {
    CUtensorMap a_re, a_im, b_re, b_im;
};

// lo = rne_tf32(x - trunc_tf32(x)) as raw bits (round to nearest on the 13 dropped bits, ties away; an exponent carry is the
// correct rounding)
__device__ __forceinline__ uint32_t split_lo(uint32_t x) {
    const float d = __uint_as_float(x) - __uint_as_float(x & 0xffffe000u);
    return (__float_as_uint(d) + 0x1000u) & 0xffffe000u;
}

__global__ void __launch_bounds__(X3_NT, 1)
    cgemm3x_kernel(const __grid_constant__ X3Maps maps, int M, int N, int K, float alpha, float beta, float *__restrict__ Cre,
                   float *__restrict__ Cim, long ldc) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + X3_STAGES * X3_STAGE);
    uint64_t *split = full + X3_STAGES;
    uint64_t *empty = split + X3_STAGES;
    uint64_t *tmem_full = empty + X3_STAGES;   // [X3_ACC]
    uint64_t *tmem_empty = tmem_full + X3_ACC;  // [X3_ACC]
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tmem_empty + X3_ACC);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tiles_m = (M + X3_BM - 1) / X3_BM, tiles_n = (N + X3_BN - 1) / X3_BN;
    const int ntiles = tiles_m * tiles_n;
    const int nk = (K + X3_KC - 1) / X3_KC;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&maps.a_re);
        tma_prefetch_desc(&maps.a_im);
        tma_prefetch_desc(&maps.b_re);
        tma_prefetch_desc(&maps.b_im);
        for (int s = 0; s < X3_STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&split[s], 4);   // one arrival per splitter warp
            mbar_init(&empty[s], 1);
        }
        for (int a = 0; a < X3_ACC; ++a) {
            mbar_init(&tmem_full[a], 1);
            mbar_init(&tmem_empty[a], 4);  // one arrival per epilogue warp
        }
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc<X3_TMEM>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    pdl_wait();
    pdl_trigger();

    // Persistent: every CTA walks the rasterised tile sequence blockIdx.x, + gridDim.x, ...; the shared-memory ring runs on
    // across tiles (iteration counter `it`), the accumulators alternate between the two halves of TMEM so that the epilogue
    // of one tile overlaps the main loop of the next.
    if (warp == 0) {
        if (lane == 0) {
            long it = 0;
            for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
                int tm, tn;
                raster(t, tiles_m, tiles_n, 12, tm, tn);
                const int m0 = tm * X3_BM, n0 = tn * X3_BN;
                for (int kt = 0; kt < nk; ++kt, ++it) {
                    const int s = (int)(it % X3_STAGES);
                    const uint32_t ph = (uint32_t)(it / X3_STAGES) & 1;
                    mbar_wait(&empty[s], ph ^ 1);
                    mbar_expect_tx(&full[s], X3_HALF);
                    unsigned char *st = smem + s * X3_STAGE;
                    const int k0 = kt * X3_KC;
#pragma unroll
                    for (int c = 0; c < X3_BM / 32; ++c) {
                        tma_load_2d(st + c * (X3_KC * 128), &maps.a_re, &full[s], m0 + 32 * c, k0);
                        tma_load_2d(st + X3_A_PLANE + c * (X3_KC * 128), &maps.a_im, &full[s], m0 + 32 * c, k0);
                    }
                    tma_load_2d(st + 2 * X3_A_PLANE, &maps.b_re, &full[s], k0, n0);
                    tma_load_2d(st + 2 * X3_A_PLANE + X3_B_PLANE, &maps.b_im, &full[s], k0, n0);
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            constexpr uint32_t ID = idesc_tf32(X3_BM, X3_BN, 1, 0, 0, 0);
            constexpr uint32_t ID_NEGA = idesc_tf32(X3_BM, X3_BN, 1, 0, 1, 0);
            long it = 0;
            int ti = 0;
            for (int t = blockIdx.x; t < ntiles; t += gridDim.x, ++ti) {
                const int a = ti % X3_ACC;
                const uint32_t aph = (uint32_t)(ti / X3_ACC) & 1;
                mbar_wait(&tmem_empty[a], aph ^ 1);  // the epilogue of tile ti - X3_ACC has drained this accumulator
                tc_fence_after();
                const uint32_t d_re = tmem + (uint32_t)(a * 2 * X3_BN), d_im = d_re + X3_BN;
                for (int kt = 0; kt < nk; ++kt, ++it) {
                    const int s = (int)(it % X3_STAGES);
                    const uint32_t ph = (uint32_t)(it / X3_STAGES) & 1;
                    mbar_wait(&split[s], ph);
                    tc_fence_after();
                    const uint32_t base = smem_u32(smem + s * X3_STAGE);
#pragma unroll
                    for (int ks = 0; ks < X3_KC / 8; ++ks) {
                        // part p = 0: hi tiles, 1: lo tiles (same layout X3_HALF further on)
                        uint64_t dar[2], dai[2], dbr[2], dbi[2];
#pragma unroll
                        for (int p = 0; p < 2; ++p) {
                            const uint32_t a_re = base + p * X3_HALF, a_im = a_re + X3_A_PLANE;
                            const uint32_t b_re = a_re + 2 * X3_A_PLANE, b_im = b_re + X3_B_PLANE;
                            dar[p] = smem_desc_sw128_base32(a_re + ks * 1024, X3_KC * 128, 512);
                            dai[p] = smem_desc_sw128_base32(a_im + ks * 1024, X3_KC * 128, 512);
                            dbr[p] = smem_desc_sw64(b_re + ks * 32, 16, 512);
                            dbi[p] = smem_desc_sw64(b_im + ks * 32, 16, 512);
                        }
                        // the two small terms first, then hi*hi: (a, b) part pairs (1,0), (0,1), (0,0)
#pragma unroll
                        for (int tt = 0; tt < 3; ++tt) {
                            const int pa = tt == 0 ? 1 : 0, pb = tt == 1 ? 1 : 0;
                            const uint32_t acc = (kt | ks | tt) ? 1u : 0u;
                            umma_tf32(d_re, dar[pa], dbr[pb], ID, acc);        // Dr += Ar Br
                            umma_tf32(d_im, dar[pa], dbi[pb], ID, acc);        // Di += Ar Bi
                            umma_tf32(d_re, dai[pa], dbi[pb], ID_NEGA, 1u);    // Dr -= Ai Bi
                            umma_tf32(d_im, dai[pa], dbr[pb], ID, 1u);         // Di += Ai Br
                        }
                    }
                    umma_commit(&empty[s]);
                }
                umma_commit(&tmem_full[a]);
            }
        }
    } else if (warp >= 6) {
        // ---- splitters: lo at +X3_HALF from the landed words, 16 bytes at a time
        const int tid = threadIdx.x - 192;  // 0 .. 127
        long it = 0;
        for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
            for (int kt = 0; kt < nk; ++kt, ++it) {
                const int s = (int)(it % X3_STAGES);
                const uint32_t ph = (uint32_t)(it / X3_STAGES) & 1;
                mbar_wait(&full[s], ph);
                uint4 *hi = reinterpret_cast<uint4 *>(smem + s * X3_STAGE);
                uint4 *lo = reinterpret_cast<uint4 *>(smem + s * X3_STAGE + X3_HALF);
#pragma unroll 4
                for (int i = tid; i < X3_HALF / 16; i += 128) {
                    const uint4 x = hi[i];
                    uint4 l;
                    l.x = split_lo(x.x);
                    l.y = split_lo(x.y);
                    l.z = split_lo(x.z);
                    l.w = split_lo(x.w);
                    lo[i] = l;
                }
                fence_proxy_async();  // the UMMAs (async proxy) must see these generic-proxy writes
                __syncwarp();
                if (lane == 0) mbar_arrive(&split[s]);
            }
        }
    } else {
        const int q = warp & 3;
        int ti = 0;
        for (int t = blockIdx.x; t < ntiles; t += gridDim.x, ++ti) {
            const int a = ti % X3_ACC;
            const uint32_t aph = (uint32_t)(ti / X3_ACC) & 1;
            int tm, tn;
            raster(t, tiles_m, tiles_n, 12, tm, tn);
            const int n0 = tn * X3_BN;
            const long row = (long)tm * X3_BM + 32 * q + lane;
            const bool row_ok = row < M;
            mbar_wait(&tmem_full[a], aph);
            tc_fence_after();
            const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16) + (uint32_t)(a * 2 * X3_BN);
            // the old C values of chunk i + 1 are requested before chunk i is stored
            float oldr[2][16], oldi[2][16];
            auto load_old = [&](int c0, float (&orr)[16], float (&oii)[16]) {
                if (beta == 0.f) return;
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const long col = (long)n0 + c0 + j;
                    const bool ok = row_ok && col < N;
                    orr[j] = ok ? Cre[col * ldc + row] : 0.f;
                    oii[j] = ok ? Cim[col * ldc + row] : 0.f;
                }
            };
            load_old(0, oldr[0], oldi[0]);
#pragma unroll
            for (int ci = 0; ci < X3_BN / 16; ++ci) {
                const int c0 = 16 * ci;
                if (n0 + c0 >= N) break;  // warp-uniform
                uint32_t ar[16], ai[16];
                if (nk > 0) {
                    tmem_ld16(lane_base + c0, ar);
                    tmem_ld16(lane_base + X3_BN + c0, ai);
                }
                if (ci + 1 < X3_BN / 16) load_old(c0 + 16, oldr[(ci + 1) & 1], oldi[(ci + 1) & 1]);
                if (nk > 0) {
                    tmem_ld_wait();
                } else {
#pragma unroll
                    for (int j = 0; j < 16; ++j) ar[j] = ai[j] = 0u;
                }
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const long col = (long)n0 + c0 + j;
                    if (row_ok && col < N) {
                        float vr = alpha * __uint_as_float(ar[j]), vi = alpha * __uint_as_float(ai[j]);
                        if (beta != 0.f) {
                            vr = fmaf(beta, oldr[ci & 1][j], vr);
                            vi = fmaf(beta, oldi[ci & 1][j], vi);
                        }
                        Cre[col * ldc + row] = vr;
                        Cim[col * ldc + row] = vi;
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&tmem_empty[a]);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc<X3_TMEM>(tmem);
}

}  // namespace

// FP32-class planar complex64 GEMM on tcgen05.  C must not alias A or B.  Same argument rules as cgemm (cgemm.cu).
int cgemm3x(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C) {
    if (m <= 0 || n <= 0) return 0;
    if (k <= 0 && beta == 1.0) return 0;
    if (((uintptr_t)A.re | (uintptr_t)A.im | (uintptr_t)B.re | (uintptr_t)B.im) & 15) return -6;
    if ((A.ld | B.ld) & 3) return -7;
    auto kern = cgemm3x_kernel;
    static SmemCfg cfg;
    HP_TRY(configure_smem(cfg, kern, X3_SMEM));
    X3Maps maps;
    const int kk = k > 0 ? k : 1;
    HP_TRY(make_map(&maps.a_re, A.re, m, kk, A.ld, 32, X3_KC, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B));
    HP_TRY(make_map(&maps.a_im, A.im, m, kk, A.ld, 32, X3_KC, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B));
    HP_TRY(make_map(&maps.b_re, B.re, kk, n, B.ld, X3_KC, X3_BN, CU_TENSOR_MAP_SWIZZLE_64B));
    HP_TRY(make_map(&maps.b_im, B.im, kk, n, B.ld, X3_KC, X3_BN, CU_TENSOR_MAP_SWIZZLE_64B));
    const bool prof = prof_enabled() && k > 0;
    if (prof) prof_begin(st, 8.0 * m * n * k);
    const long ntiles = (long)ceil_div(m, X3_BM) * ceil_div(n, X3_BN);
    HP_CUDA(launch_pdl(kern, dim3((unsigned)std::min<long>(ntiles, kNumSMs)), dim3(X3_NT), X3_SMEM, st, maps, m, n, k, (float)alpha,
                       (float)beta, C.re, C.im, (long)C.ld));
    if (prof) prof_end(st);
    HP_LAUNCHED();
    return 0;
}

// The FP32-class product the factorisation and the solves call: the tcgen05 kernel when the operands are distinct and the
// problem fills tiles, else the mma.sync kernel (cgemm3.cu: in-place leaves, tiny shapes).  variant: 0 auto, 1 mma.sync
// always, 2 tcgen05 whenever legal (tests, A/B timing).
static std::atomic<int> g_c3_variant{0};
int cgemm3_any(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C) {
    const int v = g_c3_variant.load(std::memory_order_relaxed);
    const bool distinct = C.re != A.re && C.re != B.re && C.im != A.im && C.im != B.im;
    const bool legal = distinct && k > 0;
    const bool worth = m >= 128 && n >= 32 && k >= 64 && (long)ceil_div(m, X3_BM) * ceil_div(n, X3_BN) >= 32;
    if (legal && v != 1 && (v == 2 || worth)) return cgemm3x(st, m, n, k, alpha, A, B, beta, C);
    return cgemm3(st, m, n, k, alpha, A, B, beta, C);
}

}  // namespace hp

extern "C" int hprmat_profile_cgemm3_variant(int v) {
    if (v < 0 || v > 2) return -1;
    hp::g_c3_variant.store(v, std::memory_order_relaxed);
    return 0;
}
