// zgemm3m.cu -- complex128 GEMM on the FP64 tensor cores in the "3M" real decomposition (north_star: "3M or 4M real
// decomposition chosen by measurement"):
//
//   C <- beta*C + alpha*A*B,   A m x k, B k x n, C m x n, interleaved complex128, column-major.
//
// With A = Ar + i Ai, B = Br + i Bi:   T1 = Ar Br,  T2 = Ai Bi,  T3 = (Ar + Ai)(Br + Bi)
//                                      Re(AB) = T1 - T2,   Im(AB) = T3 - T1 - T2
// i.e. three real products instead of the four of zgemm.cu (25 % fewer DMMAs for the same complex product); the sums
// Ar + Ai, Br + Bi are formed in registers on the fragments (one DADD per fragment element).  The imaginary part is only
// NORMWISE accurate, |err| <~ u (|Ar| + |Ai|)(|Br| + |Bi|): that is the error model of the LU's backward error anyway, and the
// refinement of the R-matrix path does not see it.  Flop accounting: the paper's convention (8 per complex multiply-add)
// is kept for the reported TFLOP/s; the HARDWARE flops of this kernel are 6 m n k, and roofline fractions use those.
//
// One mma.sync.m8n8k4.f64 = 8 x 8 real outputs over 4 real k = here 8 complex rows x 8 columns x 4 complex k of ONE of the
// three products.  A fragment: lane (r = lane/4, kk = lane%4) holds element (row r, k kk): one LDS.128 fetches (re, im) of
// that complex element; same for B with (k kk, col r).  C fragment: lane holds (row r, cols 2kk, 2kk+1) of T1, T2, T3, so
// the complex result of an element is combined inside one lane and stored as one 16-byte word.
// Tiling: CTA = WM x WN warps, warp tile 32 x 16 (4 x 2 MMA tiles, 3 accumulators each = 96 registers), k-slab KC,
// cp.async ring synchronised by mbarriers (no CTA-wide barrier in the main loop); shared leading dimensions BM + 2 (A stored [k][m]) and KC + 4 (B stored [n][k]) make the 16-byte fragment
// loads conflict free.  C may NOT alias B here (several M tiles per column strip): zgemm() routes such calls to zgemm.cu.
#include "lu.cuh"
#include "sm100.cuh"

namespace hp {

namespace {

using namespace sm100;

__device__ __forceinline__ void cp16(void *sdst, const void *gsrc, bool valid) {
    unsigned s = (unsigned)__cvta_generic_to_shared(sdst);
    int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gsrc), "r"(sz) : "memory");
}
// the mbarrier receives one arrival when all cp.async issued so far by this thread have landed
__device__ __forceinline__ void cp_arrive_noinc(uint64_t *bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

template <int WM, int WN, int KC, int STAGES, int LP>
__global__ void __launch_bounds__(WM *WN * 32, 1)
    zgemm3m_kernel(int M, int N, int K, double alpha, const double2 *__restrict__ A, long lda, const double2 *__restrict__ B,
                   long ldb, double beta, double2 *__restrict__ C, long ldc, long strideA, long strideB, long strideC) {
    constexpr int BM = WM * 32, BN = WN * 16, NT = WM * WN * 32;
    constexpr int LDA_S = BM + 2, LDB_S = KC + 4;
    constexpr int A_STAGE = KC * LDA_S, B_STAGE = BN * LDB_S;
    static_assert(KC % 4 == 0, "KC must be a multiple of 4");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *sA = reinterpret_cast<double2 *>(smem_raw);
    double2 *sB = sA + STAGES * A_STAGE;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int wm = warp % WM, wn = warp / WM;
    const int r = lane >> 2, kk = lane & 3;
    int tm, tn;
    raster((int)blockIdx.x, (M + BM - 1) / BM, (N + BN - 1) / BN, 16, tm, tn);
    const long m0 = (long)tm * BM, n0 = (long)tn * BN;
    A += (long)blockIdx.z * strideA;
    B += (long)blockIdx.z * strideB;
    C += (long)blockIdx.z * strideC;

    auto load_stage = [&](int slot, int k0) {
        double2 *a = sA + slot * A_STAGE;
        double2 *b = sB + slot * B_STAGE;
#pragma unroll
        for (int idx = tid; idx < BM * KC; idx += NT) {
            const int i = idx % BM, p = idx / BM;
            const bool ok = (m0 + i < M) && (k0 + p < K);
            cp16(a + p * LDA_S + i, ok ? (A + (long)(k0 + p) * lda + m0 + i) : A, ok);
        }
#pragma unroll
        for (int idx = tid; idx < BN * KC; idx += NT) {
            const int p = idx % KC, n = idx / KC;
            const bool ok = (n0 + n < N) && (k0 + p < K);
            cp16(b + n * LDB_S + p, ok ? (B + (n0 + n) * ldb + k0 + p) : B, ok);
        }
    };

    double t1[4][2][2], t2[4][2][2], t3[4][2][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) t1[i][j][e] = t2[i][j][e] = t3[i][j][e] = 0.0;

    const int nk = (K + KC - 1) / KC;
    // No CTA-wide barrier in the main loop.  full[s] (NT arrivals, one per thread when its cp.async of the stage have landed)
    // releases the readers of a stage; empty[s] (one arrival per warp) releases its slot for the load of slab kt + STAGES - 1,
    // which is issued at k-step LP of slab kt -- most of a slab after every warp has left slab kt - 1, so neither wait is
    // reached before its condition holds unless the warps drift apart by that much.  (The position of the issue point
    // matters by itself: +4 % at LP = 6 against LP = 0, 2 or 5, profiles/r01_ncu_full.md.)
    __shared__ uint64_t full_bar[STAGES], empty_bar[STAGES];
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(&full_bar[s], NT);
            mbar_init(&empty_bar[s], WM * WN);
        }
        fence_mbar_init();
    }
    __syncthreads();
    pdl_wait();
    pdl_trigger();
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nk) {
            load_stage(s, s * KC);
            cp_arrive_noinc(&full_bar[s]);
        }
    }
    const int a_off = kk * LDA_S + wm * 32 + r;       // + ks*4*LDA_S + mi*8
    const int b_off = (wn * 16 + r) * LDB_S + kk;     // + ni*8*LDB_S + ks*4

    for (int kt = 0; kt < nk; ++kt) {
        mbar_wait(&full_bar[kt % STAGES], (kt / STAGES) & 1);
        const double2 *a_s = sA + (kt % STAGES) * A_STAGE + a_off;
        const double2 *b_s = sB + (kt % STAGES) * B_STAGE + b_off;
        // Software pipeline over the k-steps: the fragments of step ks + 1 are fetched before the MMAs of step ks are issued,
        // and their sums (DADDs, which queue on the same FP64 pipe as the DMMAs) are formed after them, a whole step before use.
        double2 af[2][4], bf[2][2];
        double as[2][4], bs[2][2];
        auto fetch = [&](int ks, int b) {
#pragma unroll
            for (int mi = 0; mi < 4; ++mi) af[b][mi] = a_s[ks * 4 * LDA_S + mi * 8];
#pragma unroll
            for (int ni = 0; ni < 2; ++ni) bf[b][ni] = b_s[ni * 8 * LDB_S + ks * 4];
        };
        auto sums = [&](int b) {
#pragma unroll
            for (int mi = 0; mi < 4; ++mi) as[b][mi] = af[b][mi].x + af[b][mi].y;
#pragma unroll
            for (int ni = 0; ni < 2; ++ni) bs[b][ni] = bf[b][ni].x + bf[b][ni].y;
        };
        fetch(0, 0);
        sums(0);
#pragma unroll
        for (int ks = 0; ks < KC / 4; ++ks) {
            const int b = ks & 1;
            if (ks == LP) {
                const int nxt = kt + STAGES - 1;
                if (nxt < nk) {
                    const int ps = nxt % STAGES;  // the slot of slab kt - 1
                    if (nxt >= STAGES) mbar_wait(&empty_bar[ps], ((nxt / STAGES) - 1) & 1);
                    load_stage(ps, nxt * KC);
                    cp_arrive_noinc(&full_bar[ps]);
                }
            }
            if (ks + 1 < KC / 4) fetch(ks + 1, b ^ 1);
#pragma unroll
            for (int mi = 0; mi < 4; ++mi)
#pragma unroll
                for (int ni = 0; ni < 2; ++ni) {
                    dmma(t1[mi][ni], af[b][mi].x, bf[b][ni].x);
                    dmma(t2[mi][ni], af[b][mi].y, bf[b][ni].y);
                }
#pragma unroll
            for (int mi = 0; mi < 4; ++mi)
#pragma unroll
                for (int ni = 0; ni < 2; ++ni) dmma(t3[mi][ni], as[b][mi], bs[b][ni]);
            if (ks + 1 < KC / 4) sums(b ^ 1);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[kt % STAGES]);
    }

    // epilogue: element (row 8 mi + r, col 8 ni + 2 kk + e) of the warp tile; old C values fetched as independent loads first
    double2 old[4][2][2];
    if (beta != 0.0) {
#pragma unroll
        for (int mi = 0; mi < 4; ++mi)
#pragma unroll
            for (int ni = 0; ni < 2; ++ni)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const long row = m0 + wm * 32 + mi * 8 + r, col = n0 + wn * 16 + ni * 8 + 2 * kk + e;
                    old[mi][ni][e] = (row < M && col < N) ? C[col * ldc + row] : make_double2(0.0, 0.0);
                }
    }
#pragma unroll
    for (int mi = 0; mi < 4; ++mi)
#pragma unroll
        for (int ni = 0; ni < 2; ++ni)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const long row = m0 + wm * 32 + mi * 8 + r, col = n0 + wn * 16 + ni * 8 + 2 * kk + e;
                if (row < M && col < N) {
                    double vr = alpha * (t1[mi][ni][e] - t2[mi][ni][e]);
                    double vi = alpha * ((t3[mi][ni][e] - t1[mi][ni][e]) - t2[mi][ni][e]);
                    if (beta != 0.0) {
                        vr += beta * old[mi][ni][e].x;
                        vi += beta * old[mi][ni][e].y;
                    }
                    C[col * ldc + row] = make_double2(vr, vi);
                }
            }
}

}  // namespace

int zgemm3m(cudaStream_t st, int m, int n, int k, double alpha, const double2 *A, long lda, long strideA, const double2 *B,
            long ldb, long strideB, double beta, double2 *C, long ldc, long strideC, int nbatch) {
    constexpr int WM = 2, WN = 4, KC = 32, STAGES = 3;
    constexpr int BM = WM * 32, BN = WN * 16;
    constexpr size_t smem = (size_t)STAGES * (KC * (BM + 2) + BN * (KC + 4)) * sizeof(double2);
    constexpr int LP = 6;
    static_assert(LP < KC / 4, "the issue point is a k-step of the slab");
    auto kern = zgemm3m_kernel<WM, WN, KC, STAGES, LP>;
    static SmemCfg cfg;
    HP_TRY(configure_smem(cfg, kern, smem));
    dim3 grid(ceil_div(m, BM) * ceil_div(n, BN), 1, nbatch);
    HP_CUDA(launch_pdl(kern, grid, dim3(WM * WN * 32), smem, st, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, strideA, strideB,
                       strideC));
    HP_LAUNCHED();
    return 0;
}

}  // namespace hp
