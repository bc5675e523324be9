// cgemm_splitk.cu -- planar complex64 GEMM on tcgen05 (kind::tf32) for products with FEW output tiles and a DEEP inner
// dimension: the forward / backward substitutions of the mixed modes ("forward and backward
// substitution" for the Nc right-hand sides) in their left-looking form, B_k -= L[k, 0:k] Y[0:k], and the products with the
// kept block inverses -- 1024 x Nc outputs (16 tiles at Nc = 256) against an inner dimension of up to N.
//
//   C <- beta*C + alpha*A*B,  same operand layouts and arithmetic as cgemm.cu.
//
// One 128 x 128 output tile is computed by a CLUSTER of S CTAs (S <= 8), each accumulating one slice of K in its own TMEM;
// the S partial tiles are then reduced through DISTRIBUTED SHARED MEMORY in a fixed order (deterministic, no atomics):
// every CTA parks its partial tile in its own shared memory (the operand ring is free by then), the cluster synchronises,
// and CTA r sums rows [128 r / S, 128 (r+1) / S) of all S partials with ld.shared::cluster, applies alpha / beta and writes
// that strip of C.  16 tiles x 8 slices = 128 CTAs: one wave of the GPU instead of 16 busy SMs.
#include "lu.cuh"
#include "sm100.cuh"

namespace hp {

using namespace sm100;

int make_map(CUtensorMap *map, const float *plane, long rows, long cols, long ld, int box_rows, int box_cols,
             CUtensorMapSwizzle swz);  // cgemm.cu

namespace {

constexpr int SK_BM = 128, SK_BN = 128, SK_KC = 32, SK_NT = 192;
constexpr int SK_A_PLANE = SK_BM * SK_KC * 4, SK_B_PLANE = SK_BN * SK_KC * 4;
constexpr int SK_STAGE = 2 * SK_A_PLANE + 2 * SK_B_PLANE;  // 64 KB
constexpr int SK_STAGES = 3;
constexpr int SK_SMEM = SK_STAGES * SK_STAGE + 1024 + 256;
constexpr int SK_TMEM = 2 * SK_BN;
constexpr int SK_PLD = SK_BM + 4;  // column stride (floats) of the parked partial tile: rows contiguous, columns skewed by 16 B

struct SkMaps {
    CUtensorMap a_re, a_im, b_re, b_im;
};

__device__ __forceinline__ uint32_t cluster_nctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;\n" : "=r"(r));
    return r;
}
// not volatile: the loads of all slices of a chunk are independent and must be in flight together (DSMEM latency ~0.1 us)
__device__ __forceinline__ float4 ld_cluster_f4(uint32_t addr) {
    float4 v;
    asm("ld.shared::cluster.v4.f32 {%0,%1,%2,%3}, [%4];\n" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}

template <int S>
__global__ void __launch_bounds__(SK_NT, 1)
    cgemm_splitk_kernel(const __grid_constant__ SkMaps maps, int M, int N, int K, float alpha, float beta, float *__restrict__ Cre,
                        float *__restrict__ Cim, long ldc, int tiles_m) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + SK_STAGES * SK_STAGE);
    uint64_t *empty = full + SK_STAGES;
    uint64_t *tmem_full = empty + SK_STAGES;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tmem_full + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const int tile = (int)(blockIdx.x / S);
    const int tm = tile % tiles_m, tn = tile / tiles_m;
    const int m0 = tm * SK_BM, n0 = tn * SK_BN;
    const int nk_all = (K + SK_KC - 1) / SK_KC;
    const int kt0 = (int)((long)nk_all * rank / S), kt1 = (int)((long)nk_all * (rank + 1) / S);  // this CTA's slice of K
    const int nk = kt1 - kt0;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&maps.a_re);
        tma_prefetch_desc(&maps.a_im);
        tma_prefetch_desc(&maps.b_re);
        tma_prefetch_desc(&maps.b_im);
        for (int s = 0; s < SK_STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 1);
        }
        mbar_init(tmem_full, 1);
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc<SK_TMEM>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    pdl_wait();     // the prologue above may overlap the predecessor's tail (launch_pdl); global memory only from here on
    pdl_trigger();

    if (warp == 0) {
        if (lane == 0) {
            for (int i = 0; i < nk; ++i) {
                const int s = i % SK_STAGES;
                const uint32_t ph = (i / SK_STAGES) & 1;
                mbar_wait(&empty[s], ph ^ 1);
                mbar_expect_tx(&full[s], SK_STAGE);
                unsigned char *st = smem + s * SK_STAGE;
                const int k0 = (kt0 + i) * SK_KC;
#pragma unroll
                for (int c = 0; c < SK_BM / 32; ++c) {
                    tma_load_2d(st + c * (SK_KC * 128), &maps.a_re, &full[s], m0 + 32 * c, k0);
                    tma_load_2d(st + SK_A_PLANE + c * (SK_KC * 128), &maps.a_im, &full[s], m0 + 32 * c, k0);
                }
                tma_load_2d(st + 2 * SK_A_PLANE, &maps.b_re, &full[s], k0, n0);
                tma_load_2d(st + 2 * SK_A_PLANE + SK_B_PLANE, &maps.b_im, &full[s], k0, n0);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            constexpr uint32_t ID = idesc_tf32(SK_BM, SK_BN, 1, 0, 0, 0);
            constexpr uint32_t ID_NEGA = idesc_tf32(SK_BM, SK_BN, 1, 0, 1, 0);
            const uint32_t d_re = tmem, d_im = tmem + SK_BN;
            for (int i = 0; i < nk; ++i) {
                const int s = i % SK_STAGES;
                const uint32_t ph = (i / SK_STAGES) & 1;
                mbar_wait(&full[s], ph);
                tc_fence_after();
                const uint32_t a_re = smem_u32(smem + s * SK_STAGE), a_im = a_re + SK_A_PLANE;
                const uint32_t b_re = a_re + 2 * SK_A_PLANE, b_im = b_re + SK_B_PLANE;
#pragma unroll
                for (int ks = 0; ks < SK_KC / 8; ++ks) {
                    const uint64_t dar = smem_desc_sw128_base32(a_re + ks * 1024, SK_KC * 128, 512);
                    const uint64_t dai = smem_desc_sw128_base32(a_im + ks * 1024, SK_KC * 128, 512);
                    const uint64_t dbr = smem_desc_sw128(b_re + ks * 32, 16, 1024);
                    const uint64_t dbi = smem_desc_sw128(b_im + ks * 32, 16, 1024);
                    const uint32_t acc = (i | ks) ? 1u : 0u;
                    umma_tf32(d_re, dar, dbr, ID, acc);
                    umma_tf32(d_im, dar, dbi, ID, acc);
                    umma_tf32(d_re, dai, dbi, ID_NEGA, 1u);
                    umma_tf32(d_im, dai, dbr, ID, 1u);
                }
                umma_commit(&empty[s]);
            }
            umma_commit(tmem_full);
        }
    } else {
        // ---- park this CTA's partial tile in shared memory: part[plane][col][row], row = TMEM lane (conflict-free)
        const int q = warp & 3;
        const int row = 32 * q + lane;
        float *part = reinterpret_cast<float *>(smem);
        mbar_wait(tmem_full, 0);  // all MMAs done, hence all operand loads consumed: the ring is free
        tc_fence_after();
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
#pragma unroll 1
        for (int c0 = 0; c0 < SK_BN; c0 += 16) {
            uint32_t ar[16], ai[16];
            if (nk > 0) {
                tmem_ld16(lane_base + c0, ar);
                tmem_ld16(lane_base + SK_BN + c0, ai);
                tmem_ld_wait();
            } else {
#pragma unroll
                for (int j = 0; j < 16; ++j) ar[j] = ai[j] = 0u;
            }
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                part[(size_t)(c0 + j) * SK_PLD + row] = __uint_as_float(ar[j]);
                part[(size_t)(SK_BN + c0 + j) * SK_PLD + row] = __uint_as_float(ai[j]);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();  // every partial tile of the cluster is in shared memory
    if (warp >= 2) {
        // ---- CTA `rank` reduces the rows [r0, r1) of the tile over the S partials, in slice order
        const int t = threadIdx.x - 64;  // 0 .. 127
        const int r0 = (int)(SK_BM * rank / S), r1 = (int)(SK_BM * (rank + 1) / S);  // multiples of 4 (S = 2, 4, 8)
        const int nrc = (r1 - r0) / 4;                                               // 4-row chunks per column
        const uint32_t base = smem_u32(smem);
        for (int c = t; c < SK_BN * nrc; c += 128) {
            const int cl = c / nrc, r = r0 + 4 * (c - cl * nrc);
            const long col = (long)n0 + cl;
            float4 pr[S], pi[S];
#pragma unroll
            for (int s = 0; s < S; ++s) {  // all 2 S loads in flight, then the sums in slice order
                const uint32_t remote = mapa_u32(base, (uint32_t)s);
                pr[s] = ld_cluster_f4(remote + (uint32_t)(((size_t)cl * SK_PLD + r) * 4));
                pi[s] = ld_cluster_f4(remote + (uint32_t)(((size_t)(SK_BN + cl) * SK_PLD + r) * 4));
            }
            float4 sr = pr[0], si = pi[0];
#pragma unroll
            for (int s = 1; s < S; ++s) {
                sr.x += pr[s].x; sr.y += pr[s].y; sr.z += pr[s].z; sr.w += pr[s].w;
                si.x += pi[s].x; si.y += pi[s].y; si.z += pi[s].z; si.w += pi[s].w;
            }
            if (col < N) {
                const float vr[4] = {sr.x, sr.y, sr.z, sr.w}, vi[4] = {si.x, si.y, si.z, si.w};
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const long grow = (long)m0 + r + e;
                    if (grow < M) {
                        float xr = alpha * vr[e], xi = alpha * vi[e];
                        if (beta != 0.f) {
                            xr = fmaf(beta, Cre[col * ldc + grow], xr);
                            xi = fmaf(beta, Cim[col * ldc + grow], xi);
                        }
                        Cre[col * ldc + grow] = xr;
                        Cim[col * ldc + grow] = xi;
                    }
                }
            }
        }
    }
    cluster_sync_all();  // nobody leaves while a peer still reads its shared memory
    if (warp == 1) tmem_dealloc<SK_TMEM>(tmem);
}

}  // namespace

// C <- beta*C + alpha*A*B with every 128 x 128 tile computed by a cluster of `slices` CTAs (2, 4 or 8) along K.
// C must not alias A or B.  Same argument rules as cgemm (cgemm.cu).
int cgemm_splitk(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C, int slices) {
    if (m <= 0 || n <= 0) return 0;
    if (((uintptr_t)A.re | (uintptr_t)A.im | (uintptr_t)B.re | (uintptr_t)B.im) & 15) return -6;
    if ((A.ld | B.ld) & 3) return -7;
    if (slices != 2 && slices != 4 && slices != 8) return -10;
    static SmemCfg cfg2, cfg4, cfg8;
    HP_TRY(configure_smem(cfg2, cgemm_splitk_kernel<2>, SK_SMEM));
    HP_TRY(configure_smem(cfg4, cgemm_splitk_kernel<4>, SK_SMEM));
    HP_TRY(configure_smem(cfg8, cgemm_splitk_kernel<8>, SK_SMEM));
    SkMaps maps;
    const int kk = k > 0 ? k : 1;
    HP_TRY(make_map(&maps.a_re, A.re, m, kk, A.ld, 32, SK_KC, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B));
    HP_TRY(make_map(&maps.a_im, A.im, m, kk, A.ld, 32, SK_KC, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B));
    HP_TRY(make_map(&maps.b_re, B.re, kk, n, B.ld, SK_KC, SK_BN, CU_TENSOR_MAP_SWIZZLE_128B));
    HP_TRY(make_map(&maps.b_im, B.im, kk, n, B.ld, SK_KC, SK_BN, CU_TENSOR_MAP_SWIZZLE_128B));
    const int tiles_m = ceil_div(m, SK_BM), tiles_n = ceil_div(n, SK_BN);
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((unsigned)(tiles_m * tiles_n * slices));
    lc.blockDim = dim3(SK_NT);
    lc.dynamicSmemBytes = SK_SMEM;
    lc.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)slices;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    lc.attrs = attr;
    lc.numAttrs = pdl_enabled() ? 2 : 1;
    const float al = (float)alpha, be = (float)beta;
    if (slices == 8) HP_CUDA(cudaLaunchKernelEx(&lc, cgemm_splitk_kernel<8>, maps, m, n, k, al, be, C.re, C.im, C.ld, tiles_m));
    else if (slices == 4) HP_CUDA(cudaLaunchKernelEx(&lc, cgemm_splitk_kernel<4>, maps, m, n, k, al, be, C.re, C.im, C.ld, tiles_m));
    else HP_CUDA(cudaLaunchKernelEx(&lc, cgemm_splitk_kernel<2>, maps, m, n, k, al, be, C.re, C.im, C.ld, tiles_m));
    HP_LAUNCHED();
    return 0;
}

}  // namespace hp
