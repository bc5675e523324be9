// zgemm.cu -- complex128 GEMM on the FP64 tensor cores (DMMA, mma.sync.m8n8k4.f64) for sm_100a.
//
//   C <- beta*C + alpha*A*B,   A m x k, B k x n, C m x n, interleaved complex128, column-major.
//
// This is the trailing update A22 <- A22 - L21*U12 of the blocked LU (Eq. 5; the O(N^3) part that
// the paper hands to ZGETRF/CGETRF), and the GEMM inside the blocked triangular solves.  tcgen05.mma has no f64 kind,
// so FP64 tensor work on sm_100a is warp-level mma.sync.
//
// Complex product on a real MMA ("4M" form, 8 real flops per complex multiply-add = the 8N^3/3 convention of
// PAPER.md:190): view column-major complex C (m x n) as the real 2m x n array C~ (re/im interleaved along rows), B as
// the real 2k x n array B~, and expand A on the fly into the real 2m x 2k array
//     A~[2i  ,2p] =  Ar   A~[2i  ,2p+1] = -Ai
//     A~[2i+1,2p] =  Ai   A~[2i+1,2p+1] =  Ar
// so that C~ = A~ * B~.  The expansion happens in registers while the A fragment is read from shared memory (each lane
// picks the real or imaginary word of one complex element and flips its sign bit if needed); B~ and C~ fragments are
// the natural memory layout.  One m8n8k4 MMA = 4 complex rows x 8 columns x 2 complex k.
//
// Tiling: CTA = WM x WN warps, warp tile 32 complex rows x 32 columns (8 x 4 MMAs per 2 complex k, 64 accumulators
// per lane), CTA tile (32 WM) x (32 WN), k-slab KC, STAGES-deep cp.async ring.  Shared-memory leading dimensions are
// padded to == 2 (mod 8) complex elements so that every fragment load (LDS.64) is bank-conflict free.
#include "lu.cuh"

namespace hp {

__device__ __forceinline__ void cp_async16(void *sdst, const void *gsrc, bool valid) {
    unsigned s = (unsigned)__cvta_generic_to_shared(sdst);
    int sz = valid ? 16 : 0;  // src-size 0 => 16 bytes of zero fill, nothing is read
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gsrc), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

template <int WM, int WN, int KC, int STAGES, int MINB>
__global__ void __launch_bounds__(WM *WN * 32, MINB)
    zgemm_kernel(int M, int N, int K, double alpha, const double2 *__restrict__ A, long lda,
                 const double2 *__restrict__ B, long ldb, double beta, double2 *C, long ldc, long strideA,
                 long strideB, long strideC) {
    constexpr int BM = WM * 32, BN = WN * 32, NT = WM * WN * 32;
    constexpr int LDA_S = BM + 2, LDB_S = KC + 2;
    constexpr int A_STAGE = KC * LDA_S, B_STAGE = BN * LDB_S;
    static_assert(KC % 8 == 0, "KC must be a multiple of 8");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *sA = reinterpret_cast<double2 *>(smem_raw);
    double2 *sB = sA + STAGES * A_STAGE;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int wm = warp % WM, wn = warp / WM;
    const int r = lane >> 2, kk = lane & 3;
    int tm, tn;
    raster((int)blockIdx.x, (M + BM - 1) / BM, (N + BN - 1) / BN, 8, tm, tn);
    const long m0 = (long)tm * BM, n0 = (long)tn * BN;
    A += (long)blockIdx.z * strideA;
    B += (long)blockIdx.z * strideB;
    C += (long)blockIdx.z * strideC;
    pdl_wait();
    pdl_trigger();

    auto load_stage = [&](int slot, int k0) {
        double2 *a = sA + slot * A_STAGE;
        double2 *b = sB + slot * B_STAGE;
#pragma unroll
        for (int idx = tid; idx < BM * KC; idx += NT) {
            int i = idx % BM, p = idx / BM;
            bool ok = (m0 + i < M) && (k0 + p < K);
            const double2 *src = ok ? (A + (long)(k0 + p) * lda + m0 + i) : A;
            cp_async16(a + p * LDA_S + i, src, ok);
        }
#pragma unroll
        for (int idx = tid; idx < BN * KC; idx += NT) {
            int p = idx % KC, n = idx / KC;
            bool ok = (n0 + n < N) && (k0 + p < K);
            const double2 *src = ok ? (B + (n0 + n) * ldb + k0 + p) : B;
            cp_async16(b + n * LDB_S + p, src, ok);
        }
    };

    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const int nk = (K + KC - 1) / KC;
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nk) load_stage(s, s * KC);
        cp_async_commit();
    }

    // per-lane fragment offsets (in doubles) inside a stage
    const int a_off0 = ((kk >> 1) * LDA_S + wm * 32 + (r >> 1)) * 2 + ((r ^ kk) & 1);
    const int b_off0 = ((wn * 32 + r) * LDB_S) * 2 + kk;
    const unsigned sign_hi = (((r & 1) == 0) && ((kk & 1) == 1)) ? 0x80000000u : 0u;

    for (int kt = 0; kt < nk; ++kt) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            int nxt = kt + STAGES - 1;
            if (nxt < nk) load_stage(nxt % STAGES, nxt * KC);
            cp_async_commit();
        }
        const int slot = kt % STAGES;
        const double *a_s = reinterpret_cast<const double *>(sA + slot * A_STAGE) + a_off0;
        const double *b_s = reinterpret_cast<const double *>(sB + slot * B_STAGE) + b_off0;
        // fragments of k-step ks + 1 are fetched (and the A signs applied) before the MMAs of k-step ks are issued
        double af[2][8], bf[2][4];
        auto load_frags = [&](int ks, int buf) {
#pragma unroll
            for (int ai = 0; ai < 8; ++ai) {
                double v = a_s[ks * (2 * LDA_S * 2) + ai * 8];
                int hi = __double2hiint(v) ^ (int)sign_hi;
                af[buf][ai] = __hiloint2double(hi, __double2loint(v));
            }
#pragma unroll
            for (int bi = 0; bi < 4; ++bi) bf[buf][bi] = b_s[ks * 4 + bi * (8 * LDB_S * 2)];
        };
        load_frags(0, 0);
#pragma unroll
        for (int ks = 0; ks < KC / 2; ++ks) {
            if (ks + 1 < KC / 2) load_frags(ks + 1, (ks + 1) & 1);
#pragma unroll
            for (int ai = 0; ai < 8; ++ai)
#pragma unroll
                for (int bi = 0; bi < 4; ++bi) dmma884(acc[ai][bi][0], acc[ai][bi][1], af[ks & 1][ai], bf[ks & 1][bi]);
        }
    }
    cp_async_wait<0>();

    // epilogue: lane holds C~[real row 8*ai + r][cols 8*bi + 2*kk + {0,1}] of the warp tile.  The old values of C are
    // fetched in batches of 16 independent loads before the corresponding stores (a load-store-load-store chain would
    // pay one L2 round trip per element: ~25 us per tile).
    double *Cd = reinterpret_cast<double *>(C);
#pragma unroll
    for (int ap = 0; ap < 8; ap += 2) {
        double old[2][4][2];
        if (beta != 0.0) {
#pragma unroll
            for (int a2 = 0; a2 < 2; ++a2) {
                const long crow = m0 + wm * 32 + (ap + a2) * 4 + (r >> 1);
#pragma unroll
                for (int bi = 0; bi < 4; ++bi)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const long col = n0 + wn * 32 + bi * 8 + 2 * kk + e;
                        old[a2][bi][e] = (crow < M && col < N) ? Cd[(col * ldc + crow) * 2 + (r & 1)] : 0.0;
                    }
            }
        }
#pragma unroll
        for (int a2 = 0; a2 < 2; ++a2) {
            const long crow = m0 + wm * 32 + (ap + a2) * 4 + (r >> 1);
            if (crow >= M) continue;
#pragma unroll
            for (int bi = 0; bi < 4; ++bi)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const long col = n0 + wn * 32 + bi * 8 + 2 * kk + e;
                    if (col < N) {
                        double v = alpha * acc[ap + a2][bi][e];
                        if (beta != 0.0) v += beta * old[a2][bi][e];
                        Cd[(col * ldc + crow) * 2 + (r & 1)] = v;
                    }
                }
        }
    }
}

template <int WM, int WN, int KC, int STAGES, int MINB>
static int launch_zgemm(cudaStream_t st, int m, int n, int k, double alpha, const double2 *A, long lda,
                        const double2 *B, long ldb, double beta, double2 *C, long ldc, long sA = 0, long sB = 0,
                        long sC = 0, int nbatch = 1) {
    constexpr int BM = WM * 32, BN = WN * 32;
    constexpr size_t smem = (size_t)STAGES * (KC * (BM + 2) + BN * (KC + 2)) * sizeof(double2);
    auto kern = zgemm_kernel<WM, WN, KC, STAGES, MINB>;
    static SmemCfg cfg;
    HP_TRY(configure_smem(cfg, kern, smem));
    dim3 grid(ceil_div(m, BM) * ceil_div(n, BN), 1, nbatch);
    HP_CUDA(launch_pdl(kern, grid, dim3(WM * WN * 32), smem, st, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, sA, sB, sC));
    HP_LAUNCHED();
    return 0;
}

// 3M variant (zgemm3m.cu) and the switch between the two decompositions (hprmat_zgemm_algo)
int zgemm3m(cudaStream_t st, int m, int n, int k, double alpha, const double2 *A, long lda, long strideA, const double2 *B,
            long ldb, long strideB, double beta, double2 *C, long ldc, long strideC, int nbatch);
static std::atomic<int> g_zgemm_algo{3};       // process default (hprmat_zgemm_algo)
static thread_local int tl_zgemm_algo = 0;     // a context's own setting while one of its calls runs on this thread
int zgemm_algo_in_force() { return tl_zgemm_algo ? tl_zgemm_algo : g_zgemm_algo.load(std::memory_order_relaxed); }
ScopedZgemmAlgo::ScopedZgemmAlgo(int algo) : prev(tl_zgemm_algo) {
    if (algo == 3 || algo == 4) tl_zgemm_algo = algo;
}
ScopedZgemmAlgo::~ScopedZgemmAlgo() { tl_zgemm_algo = prev; }
// the 3M kernel has several M tiles per column strip (C must not alias B) and 64-column tiles
static inline bool use_3m(int n, int k, const double2 *B, const double2 *C) {
    return zgemm_algo_in_force() == 3 && n > 32 && k >= 16 && (const void *)B != (const void *)C;
}

// C <- beta*C + alpha*A*B  (device pointers, column-major)
int zgemm(cudaStream_t st, int m, int n, int k, double alpha, const double2 *A, long lda, const double2 *B, long ldb,
          double beta, double2 *C, long ldc) {
    if (m <= 0 || n <= 0) return 0;
    if (k <= 0 && beta == 1.0) return 0;
    if (use_3m(n, k, B, C)) return zgemm3m(st, m, n, k, alpha, A, lda, 0, B, ldb, 0, beta, C, ldc, 0, 1);
    if (n <= 32) return launch_zgemm<8, 1, 8, 4, 1>(st, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc);
    return launch_zgemm<4, 2, 16, 4, 1>(st, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc);
}

int gemm(cudaStream_t st, int m, int n, int k, double alpha, ZView A, ZView B, double beta, ZView C) {
    const bool prof = prof_enabled() && m > 0 && n > 0 && k > 0;
    if (prof) prof_begin(st, 8.0 * m * n * k);
    const int rc = zgemm(st, m, n, k, alpha, A.p, A.ld, B.p, B.ld, beta, C.p, C.ld);
    if (prof) prof_end(st);
    return rc;
}

int zgemm_batched(cudaStream_t st, int m, int n, int k, double alpha, const double2 *A, long lda, long strideA,
                  const double2 *B, long ldb, long strideB, double beta, double2 *C, long ldc, long strideC, int nbatch) {
    if (m <= 0 || n <= 0 || nbatch <= 0) return 0;
    if (use_3m(n, k, B, C)) return zgemm3m(st, m, n, k, alpha, A, lda, strideA, B, ldb, strideB, beta, C, ldc, strideC, nbatch);
    if (n <= 32)
        return launch_zgemm<8, 1, 8, 4, 1>(st, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, strideA, strideB, strideC, nbatch);
    return launch_zgemm<4, 2, 16, 4, 1>(st, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, strideA, strideB, strideC, nbatch);
}

}  // namespace hp

extern "C" int hprmat_zgemm_algo(int algo) {
    if (algo == 3 || algo == 4) hp::g_zgemm_algo.store(algo);
    return hp::g_zgemm_algo.load();
}

extern "C" int hprmat_zgemm(void *cuda_stream, int m, int n, int k, double alpha, const void *A, int lda, const void *B,
                            int ldb, double beta, void *C, int ldc) {
    if (m < 0) return -2;
    if (n < 0) return -3;
    if (k < 0) return -4;
    if (lda < (m > 1 ? m : 1)) return -7;
    if (ldb < (k > 1 ? k : 1)) return -9;
    if (ldc < (m > 1 ? m : 1)) return -12;
    return hp::zgemm((cudaStream_t)cuda_stream, m, n, k, alpha, (const double2 *)A, lda, (const double2 *)B, ldb, beta,
                     (double2 *)C, ldc);
}
