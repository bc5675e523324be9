// cgemm.cu -- split-complex (planar) complex64 GEMM on the 5th-generation tensor cores: tcgen05.mma kind::tf32 with FP32
// accumulators in TMEM, operands staged by TMA (cp.async.bulk.tensor, SWIZZLE_128B) through an mbarrier ring.
//
//   C <- beta*C + alpha*A*B,   A m x k, B k x n, C m x n, each a pair of column-major float planes (re, im).
//
// This is the trailing update A22 <- A22 - L21*U12 of the low-precision LU of the mixed path (PAPER.md:147-151 Type 2,
// :192-228 Type 4: "CGETRF in single precision"; Eq. 5) and the GEMM inside its blocked triangular solves.
//
// Complex product on a real MMA, "4M" form (8 real flops per complex multiply-add = the 8N^3/3 convention):
//     Dr  = Ar*Br + (-Ai)*Bi        Di  = Ar*Bi + Ai*Br
// The sign of the second product is the negate-A bit of the instruction descriptor, so all four products are plain
// accumulating UMMAs on the four planes as they lie in memory -- that is why the mixed path stores split complex.
//
// Operand layouts in shared memory (what the column-major planes give without any transposition):
//   A tile (BM x KC): M is the contiguous dimension  -> "MN-major" canonical layout.  For 32-bit operands the only
//                     MN-major layout the UMMA accepts is SWIZZLE_128B with a 32-byte swizzle base (layout type 1; TMA's
//                     CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B): atoms of 32 (M) x 4 (K) floats.  Loaded as BM/32 TMA boxes of
//                     32 (M) x KC (K);  LBO = KC*128 B between 32-row chunks, SBO = 512 B between 4-row K groups.
//   B tile (KC x BN): K is the contiguous dimension  -> "K-major" canonical layout, rows of KC = 32 floats (128 B),
//                     swizzle atoms of 8 rows; one TMA box of 32 (K) x BN (N);  SBO = 1024 B between 8-column groups.
// TMA zero-fills out-of-bounds elements, which takes care of ragged M, N and K edges.
//
// CTA = 10 warps: warp 0 TMA producer (one lane), warp 1 TMEM allocator + UMMA issuer (one lane), warps 2-9 epilogue (two per
// TMEM lane quarter, half of the tile's columns each: 8 instead of 4 warps is +15-25 % on the k <= 512 updates, whose
// epilogue loads are latency-bound; 16 is slower again)
// (each owns the TMEM lane quarter 32*(warp%4)): tcgen05.ld -> beta*C + alpha*acc -> coalesced global stores.
#include <algorithm>

#include "lu.cuh"
#include "sm100.cuh"

namespace hp {

using namespace sm100;

namespace {

constexpr int CG_BM = 128;   // UMMA M
constexpr int CG_KC = 32;    // floats of K per stage = one 128-byte swizzle row
constexpr int CG_EPI = 8;                 // epilogue warps: two per TMEM lane quarter, each takes half of the tile's columns
constexpr int CG_NT = 64 + 32 * CG_EPI;

template <int BN> struct CgCfg {
    static constexpr int A_PLANE = CG_BM * CG_KC * 4;               // bytes of one A plane per stage (16 KB)
    static constexpr int B_PLANE = BN * CG_KC * 4;                  // bytes of one B plane per stage
    static constexpr int STAGE = 2 * A_PLANE + 2 * B_PLANE;
    static constexpr int STAGES = BN <= 32 ? 5 : BN <= 64 ? 4 : BN <= 128 ? 3 : 2;
    static constexpr int SMEM = STAGES * STAGE + 1024 /* alignment slack */ + 256 /* barriers */;
    static constexpr int TMEM_COLS = 2 * BN;                        // Dr | Di
};

struct CgMaps {
    CUtensorMap a_re, a_im, b_re, b_im;
};

template <int BN>
__global__ void __launch_bounds__(CG_NT, 1)
    cgemm_tf32_kernel(const __grid_constant__ CgMaps maps, int M, int N, int K, float alpha, float beta, float *__restrict__ Cre,
                      float *__restrict__ Cim, long ldc) {
    typedef CgCfg<BN> Cfg;
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + Cfg::STAGES * Cfg::STAGE);
    uint64_t *empty = full + Cfg::STAGES;
    uint64_t *tmem_full = empty + Cfg::STAGES;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tmem_full + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int tm, tn;
    raster((int)blockIdx.x, (M + CG_BM - 1) / CG_BM, (N + BN - 1) / BN, 12, tm, tn);
    const int m0 = tm * CG_BM, n0 = tn * BN;
    const int nk = (K + CG_KC - 1) / CG_KC;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&maps.a_re);
        tma_prefetch_desc(&maps.a_im);
        tma_prefetch_desc(&maps.b_re);
        tma_prefetch_desc(&maps.b_im);
        for (int s = 0; s < Cfg::STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 1);
        }
        mbar_init(tmem_full, 1);
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc<Cfg::TMEM_COLS>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    pdl_wait();     // everything above overlapped the predecessor's tail; global memory only from here on
    pdl_trigger();

    if (warp == 0) {
        if (lane == 0) {
            for (int kt = 0; kt < nk; ++kt) {
                const int s = kt % Cfg::STAGES;
                const uint32_t ph = (kt / Cfg::STAGES) & 1;
                mbar_wait(&empty[s], ph ^ 1);
                mbar_expect_tx(&full[s], Cfg::STAGE);
                unsigned char *st = smem + s * Cfg::STAGE;
                const int k0 = kt * CG_KC;
#pragma unroll
                for (int c = 0; c < CG_BM / 32; ++c) {
                    tma_load_2d(st + c * (CG_KC * 128), &maps.a_re, &full[s], m0 + 32 * c, k0);
                    tma_load_2d(st + Cfg::A_PLANE + c * (CG_KC * 128), &maps.a_im, &full[s], m0 + 32 * c, k0);
                }
                tma_load_2d(st + 2 * Cfg::A_PLANE, &maps.b_re, &full[s], k0, n0);
                tma_load_2d(st + 2 * Cfg::A_PLANE + Cfg::B_PLANE, &maps.b_im, &full[s], k0, n0);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            constexpr uint32_t ID = idesc_tf32(CG_BM, BN, 1, 0, 0, 0);
            constexpr uint32_t ID_NEGA = idesc_tf32(CG_BM, BN, 1, 0, 1, 0);
            const uint32_t d_re = tmem, d_im = tmem + BN;
            for (int kt = 0; kt < nk; ++kt) {
                const int s = kt % Cfg::STAGES;
                const uint32_t ph = (kt / Cfg::STAGES) & 1;
                mbar_wait(&full[s], ph);
                tc_fence_after();
                const uint32_t a_re = smem_u32(smem + s * Cfg::STAGE), a_im = a_re + Cfg::A_PLANE;
                const uint32_t b_re = a_re + 2 * Cfg::A_PLANE, b_im = b_re + Cfg::B_PLANE;
#pragma unroll
                for (int ks = 0; ks < CG_KC / 8; ++ks) {
                    // A: 8 k-rows of 128 B = 1024 B per k-step, as two 4-row (512 B) swizzle atoms; 32-row M chunks
                    // CG_KC*128 B apart
                    const uint64_t dar = smem_desc_sw128_base32(a_re + ks * 1024, CG_KC * 128, 512);
                    const uint64_t dai = smem_desc_sw128_base32(a_im + ks * 1024, CG_KC * 128, 512);
                    // B: 8 floats of K = 32 B per k-step inside the 128-byte row; 8-column groups 1024 B apart
                    const uint64_t dbr = smem_desc_sw128(b_re + ks * 32, 16, 1024);
                    const uint64_t dbi = smem_desc_sw128(b_im + ks * 32, 16, 1024);
                    const uint32_t acc = (kt | ks) ? 1u : 0u;
                    umma_tf32(d_re, dar, dbr, ID, acc);
                    umma_tf32(d_re, dai, dbi, ID_NEGA, 1u);
                    umma_tf32(d_im, dar, dbi, ID, acc);
                    umma_tf32(d_im, dai, dbr, ID, 1u);
                }
                umma_commit(&empty[s]);
            }
            umma_commit(tmem_full);
        }
    } else {
        const int q = warp & 3;  // TMEM lane quarter this warp may access
        const long row = (long)m0 + 32 * q + lane;
        constexpr int EG = (CG_EPI / 4) < (BN / 16) ? (CG_EPI / 4) : (BN / 16);   // warps per quarter that have work
        constexpr int EC = BN / EG;                    // columns per working epilogue warp
        const int cbeg = ((warp - 2) >> 2) * EC;       // (>= BN for the idle ones: their loops are empty)
        if (nk > 0) {
            mbar_wait(tmem_full, 0);
            tc_fence_after();
        }
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        const bool row_ok = row < M;
#pragma unroll 1
        for (int c0 = cbeg; c0 < cbeg + EC && c0 < BN; c0 += 16) {
            if (n0 + c0 >= N) break;  // warp-uniform
            uint32_t ar[16], ai[16];
            if (nk > 0) {
                tmem_ld16(lane_base + c0, ar);
                tmem_ld16(lane_base + BN + c0, ai);
                tmem_ld_wait();
            } else {
#pragma unroll
                for (int j = 0; j < 16; ++j) ar[j] = ai[j] = 0u;
            }
            float oldr[16], oldi[16];
            if (beta != 0.f) {
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const long col = (long)n0 + c0 + j;
                    const bool ok = row_ok && col < N;
                    oldr[j] = ok ? Cre[col * ldc + row] : 0.f;
                    oldi[j] = ok ? Cim[col * ldc + row] : 0.f;
                }
            }
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const long col = (long)n0 + c0 + j;
                if (row_ok && col < N) {
                    float vr = alpha * __uint_as_float(ar[j]), vi = alpha * __uint_as_float(ai[j]);
                    if (beta != 0.f) {
                        vr = fmaf(beta, oldr[j], vr);
                        vi = fmaf(beta, oldi[j], vi);
                    }
                    Cre[col * ldc + row] = vr;
                    Cim[col * ldc + row] = vi;
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc<Cfg::TMEM_COLS>(tmem);
}

// ---- host side: tensor maps ---------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

}  // namespace

// plane: rows x cols floats, column-major with leading dimension ld; box = box_rows x box_cols (shared with cgemm2.cu)
int make_map(CUtensorMap *map, const float *plane, long rows, long cols, long ld, int box_rows, int box_cols,
             CUtensorMapSwizzle swz) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled entry point not found");
        return HPRMAT_ECUDA;
    }
    cuuint64_t dims[2] = {(cuuint64_t)rows, (cuuint64_t)cols};
    cuuint64_t strides[1] = {(cuuint64_t)ld * sizeof(float)};
    cuuint32_t box[2] = {(cuuint32_t)box_rows, (cuuint32_t)box_cols};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void *)plane, dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled failed (%d): rows=%ld cols=%ld ld=%ld ptr=%p", (int)r,
                 rows, cols, ld, (const void *)plane);
        return HPRMAT_ECUDA;
    }
    return 0;
}

namespace {

template <int BN>
int launch_cgemm(cudaStream_t st, int m, int n, int k, float alpha, CView A, CView B, float beta, CView C) {
    typedef CgCfg<BN> Cfg;
    auto kern = cgemm_tf32_kernel<BN>;
    static SmemCfg cfg;
    HP_TRY(configure_smem(cfg, kern, Cfg::SMEM));
    CgMaps maps;
    const int kk = k > 0 ? k : 1;
    HP_TRY(make_map(&maps.a_re, A.re, m, kk, A.ld, 32, CG_KC, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B));
    HP_TRY(make_map(&maps.a_im, A.im, m, kk, A.ld, 32, CG_KC, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B));
    HP_TRY(make_map(&maps.b_re, B.re, kk, n, B.ld, CG_KC, BN, CU_TENSOR_MAP_SWIZZLE_128B));
    HP_TRY(make_map(&maps.b_im, B.im, kk, n, B.ld, CG_KC, BN, CU_TENSOR_MAP_SWIZZLE_128B));
    dim3 grid(ceil_div(m, CG_BM) * ceil_div(n, BN));
    HP_CUDA(launch_pdl(kern, grid, dim3(CG_NT), Cfg::SMEM, st, maps, m, n, k, alpha, beta, C.re, C.im, (long)C.ld));
    HP_LAUNCHED();
    return 0;
}

}  // namespace

// C <- beta*C + alpha*A*B on split-complex float planes.  Requirements (met by every caller in lu.cu): plane base
// addresses 16-byte aligned, leading dimensions multiples of 4 floats.
// which kernel serves gemm(CView): 0 = automatic (the persistent kernel, CTA pairs when there is more than one M tile),
// 1 = the one-tile-per-CTA kernel of this file, 2 = persistent single CTAs, 3 = persistent CTA pairs.  Measurement aid
// (hprmat_profile_cgemm_variant, include/hprmat_profile.h); process-wide.
static std::atomic<int> g_cgemm_variant{0};
int cgemm_variant_in_force() { return g_cgemm_variant.load(std::memory_order_relaxed); }

static int cgemm_impl(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C, unsigned *wave_ctr);
int cgemm(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C) {
    return cgemm_impl(st, m, n, k, alpha, A, B, beta, C, nullptr);
}
int cgemm_ws(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C, unsigned *wave_ctr) {
    const bool prof = prof_enabled() && m > 0 && n > 0 && k > 0;
    if (prof) prof_begin(st, 8.0 * m * n * k);
    const int rc = cgemm_impl(st, m, n, k, alpha, A, B, beta, C, wave_ctr);
    if (prof) prof_end(st);
    return rc;
}
static int cgemm_impl(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C, unsigned *wave_ctr) {
    if (m <= 0 || n <= 0) return 0;
    if (k <= 0 && beta == 1.0) return 0;
    if (((uintptr_t)A.re | (uintptr_t)A.im | (uintptr_t)B.re | (uintptr_t)B.im) & 15) return -6;
    if ((A.ld | B.ld) & 3) return -7;
    const int variant = cgemm_variant_in_force();
    const long tiles128 = (long)ceil_div(m, CG_BM) * ceil_div(n, 128);
    if ((variant >= 2 && variant <= 4) || (variant == 0 && m > CG_BM && tiles128 >= 2L * kNumSMs)) {
        // Two waves of work or more: the persistent kernel (cgemm2.cu).  Deep K and enough tiles -> pair tiles of 256 x 256
        // (N = 256 MMAs keep the tensor pipe ~18 % busier than N = 128 ones; their un-overlapped epilogue is < 5 % of such a
        // tile); otherwise pair tiles of 256 x 128 with double-buffered accumulators (epilogue under the next main loop).
        // Crossover measured on B200 between k = 2048 and 3072 (profiles/r02_cgemm.md).
        const bool deep = k >= 2560 && (long)ceil_div(m, 256) * ceil_div(n, 256) >= 4L * (kNumSMs / 2);
        const int shape = variant == 0 ? (deep ? 2 : 1) : variant - 2;
        return cgemm2(st, m, n, k, alpha, A, B, beta, C, shape, 0.f, nullptr, wave_ctr);
    }
    // Less than two waves: one tile per CTA (no persistent-loop prologue, no cluster launch), with the tile NARROWED until the
    // grid covers most of the GPU -- a 1024 x 1024 product is 8 x 8 tiles of 128 x 128 (16 % of the SMs) but 8 x 32 of
    // 128 x 32.  C aliasing A (the in-place L21 product) needs all of n inside one tile.
    const bool in_place_a = C.re == A.re;
    // Few tiles and a deep inner dimension (substitution steps, products with the kept block inverses): a cluster of CTAs per
    // tile splits K (cgemm_splitk.cu) -- as many slices as keep the grid within one wave, at least 8 k-steps of 32 each
    if ((variant == 0 || variant == 5) && !in_place_a && C.re != B.re && n > 64) {
        // as many slices as keep the grid within one wave, at least 8 k-steps of 32 per CTA (measured on B200, kernel time:
        // 1024 x 256 x 4096: 51 us against 95 us for 16 one-tile CTAs, x 12800: 104 against 272; no gain below k ~ 1024)
        int slices = 0;
        for (int sl = 8; sl >= 2; sl /= 2)
            if (tiles128 * sl <= kNumSMs && k >= 256 * sl) { slices = sl; break; }
        if (variant == 5 && slices == 0 && k >= 64) slices = 2;
        if (slices) return cgemm_splitk(st, m, n, k, alpha, A, B, beta, C, slices);
    }
    const int natural = n <= 32 ? 32 : n <= 64 ? 64 : 128;  // narrowest tile that still holds all of n
    int bn = natural;
    if (variant == 0 && !in_place_a && tiles128 < 96) bn = std::min(natural, 2 * tiles128 >= 96 ? 64 : 32);
    if (variant == 1) bn = 128;
    if (bn == 32) return launch_cgemm<32>(st, m, n, k, (float)alpha, A, B, (float)beta, C);
    if (bn == 64) return launch_cgemm<64>(st, m, n, k, (float)alpha, A, B, (float)beta, C);
    // 128 x 256 tiles when there are enough of them to fill the GPU
    if (n >= 512 && (long)ceil_div(m, CG_BM) * ceil_div(n, 256) >= 2 * kNumSMs)
        return launch_cgemm<256>(st, m, n, k, (float)alpha, A, B, (float)beta, C);
    return launch_cgemm<128>(st, m, n, k, (float)alpha, A, B, (float)beta, C);
}

int gemm(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C) {
    const bool prof = prof_enabled() && m > 0 && n > 0 && k > 0;
    if (prof) prof_begin(st, 8.0 * m * n * k);
    const int rc = cgemm(st, m, n, k, alpha, A, B, beta, C);
    if (prof) prof_end(st);
    return rc;
}

}  // namespace hp

extern "C" int hprmat_profile_cgemm_variant(int variant) {
    if (variant >= 0 && variant <= 5) hp::g_cgemm_variant.store(variant);
    return hp::g_cgemm_variant.load();
}

extern "C" int hprmat_cgemm_tf32(void *cuda_stream, int m, int n, int k, float alpha, const float *A_re, const float *A_im,
                                 int lda, const float *B_re, const float *B_im, int ldb, float beta, float *C_re, float *C_im,
                                 int ldc) {
    if (m < 0) return -2;
    if (n < 0) return -3;
    if (k < 0) return -4;
    if (lda < (m > 1 ? m : 1) || (lda & 3)) return -8;
    if (ldb < (k > 1 ? k : 1) || (ldb & 3)) return -11;
    if (ldc < (m > 1 ? m : 1)) return -15;
    using namespace hp;
    return cgemm((cudaStream_t)cuda_stream, m, n, k, alpha, CView((float *)A_re, (float *)A_im, lda),
                 CView((float *)B_re, (float *)B_im, ldb), beta, CView(C_re, C_im, ldc));
}
