// cgemm3.cu -- split-complex (planar) complex64 GEMM with FP32-class accuracy on the TF32 tensor cores ("3xTF32"):
//
//   C <- beta*C + alpha*A*B,   A m x k, B k x n, C m x n, each a pair of column-major float planes (re, im).
//
// Every operand element x is split in registers into  hi = tf32(x)  and  lo = tf32(x - hi)  and every real product is
// accumulated as  lo*hi + hi*lo + hi*hi  (FP32 accumulators), which recovers ~2^-21 relative accuracy per product instead
// of the 2^-11 of a single TF32 pass.  This is the GEMM of the triangular solves of the mixed path (PAPER.md:147-151,
// 219-225: the correction solve with the stored low-precision factors): the right-hand sides and the solution are O(1)
// quantities whose rounding to 10 mantissa bits would otherwise cap the solve at ~1e-3 and the refinement at a factor
// ~1e-3 per step.  The O(N^3) trailing update of the factorisation stays single-pass on tcgen05 (cgemm.cu).
//
// Warp-level mma.sync.m16n8k8 (tf32 in, f32 accumulate): operands must pass through registers for the split anyway, so
// the tcgen05 shared-memory operand path has nothing to offer here.  Complex product in "4M" form on the planes:
//   Cr += Ar*Br + (-Ai)*Bi        Ci += Ar*Bi + Ai*Br
// Tiling: CTA = WM x WN warps, warp tile 32 x 32 (2 x 4 MMA tiles), k-slab KC, cp.async ring.  Shared-memory leading
// dimensions (BM + 8 for A stored [k][m], KC + 4 for B stored [n][k]) make every fragment load bank-conflict free.
// C may alias B when m <= 128 (one M tile) and beta == 0: a CTA has consumed its whole B strip before it writes.
#include "lu.cuh"

namespace hp {

namespace {

__device__ __forceinline__ void cp_async16z(void *sdst, const void *gsrc, int bytes) {
    unsigned s = (unsigned)__cvta_generic_to_shared(sdst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gsrc), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ unsigned to_tf32(float x) {
    unsigned r;
    asm("cvt.rna.tf32.f32 %0, %1;\n" : "=r"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ void split_tf32(float x, unsigned &hi, unsigned &lo) {
    hi = to_tf32(x);
    lo = to_tf32(x - __uint_as_float(hi));
}
__device__ __forceinline__ void mma_tf32(float (&c)[4], const unsigned (&a)[4], const unsigned (&b)[2]) {
    asm volatile(
        "mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}
// c += a*b with both operands split: small terms first
__device__ __forceinline__ void mma3(float (&c)[4], const unsigned (&ah)[4], const unsigned (&al)[4], const unsigned (&bh)[2],
                                     const unsigned (&bl)[2]) {
    mma_tf32(c, al, bh);
    mma_tf32(c, ah, bl);
    mma_tf32(c, ah, bh);
}

constexpr int C3_WM = 4, C3_WN = 2, C3_KC = 32, C3_STAGES = 3;
constexpr int C3_BM = C3_WM * 32, C3_BN = C3_WN * 32, C3_NT = C3_WM * C3_WN * 32;
constexpr int C3_LDA = C3_BM + 8, C3_LDB = C3_KC + 4;
constexpr int C3_A_PLANE = C3_KC * C3_LDA, C3_B_PLANE = C3_BN * C3_LDB;  // floats
constexpr int C3_STAGE = 2 * C3_A_PLANE + 2 * C3_B_PLANE;                // floats
constexpr size_t C3_SMEM = (size_t)C3_STAGES * C3_STAGE * sizeof(float);

__global__ void __launch_bounds__(C3_NT, 1)
    cgemm3_kernel(int M, int N, int K, float alpha, const float *__restrict__ Are, const float *__restrict__ Aim, long lda,
                  const float *Bre, const float *Bim, long ldb, float beta, float *Cre, float *Cim, long ldc, long strideA,
                  long strideB, long strideC) {
    extern __shared__ __align__(16) float sm3[];
    Are += (long)blockIdx.y * strideA;
    Aim += (long)blockIdx.y * strideA;
    Bre += (long)blockIdx.y * strideB;
    Bim += (long)blockIdx.y * strideB;
    Cre += (long)blockIdx.y * strideC;
    Cim += (long)blockIdx.y * strideC;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int wm = warp % C3_WM, wn = warp / C3_WM;
    const int g = lane >> 2, t = lane & 3;
    int tm, tn;
    raster((int)blockIdx.x, (M + C3_BM - 1) / C3_BM, (N + C3_BN - 1) / C3_BN, 8, tm, tn);
    const long m0 = (long)tm * C3_BM, n0 = (long)tn * C3_BN;
    pdl_wait();
    pdl_trigger();

    auto load_stage = [&](int slot, int k0) {
        float *ar = sm3 + (size_t)slot * C3_STAGE, *ai = ar + C3_A_PLANE, *br = ai + C3_A_PLANE, *bi = br + C3_B_PLANE;
        // A: KC columns of BM floats, 16-byte chunks along m
        for (int idx = tid; idx < C3_KC * (C3_BM / 4); idx += C3_NT) {
            const int p = idx / (C3_BM / 4), i4 = (idx % (C3_BM / 4)) * 4;
            const long m = m0 + i4, kk = k0 + p;
            int bytes = (kk < K && m < M) ? (int)min(16L, (M - m) * 4) : 0;
            const long off = bytes ? kk * lda + m : 0;
            cp_async16z(ar + p * C3_LDA + i4, Are + off, bytes);
            cp_async16z(ai + p * C3_LDA + i4, Aim + off, bytes);
        }
        // B: BN columns of KC floats, 16-byte chunks along k
        for (int idx = tid; idx < C3_BN * (C3_KC / 4); idx += C3_NT) {
            const int n = idx / (C3_KC / 4), p4 = (idx % (C3_KC / 4)) * 4;
            const long kk = k0 + p4, nn = n0 + n;
            int bytes = (nn < N && kk < K) ? (int)min(16L, (K - kk) * 4) : 0;
            const long off = bytes ? nn * ldb + kk : 0;
            cp_async16z(br + n * C3_LDB + p4, Bre + off, bytes);
            cp_async16z(bi + n * C3_LDB + p4, Bim + off, bytes);
        }
    };

    float cr[2][4][4], ci[2][4][4];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int e = 0; e < 4; ++e) cr[i][j][e] = ci[i][j][e] = 0.f;

    const int nk = (K + C3_KC - 1) / C3_KC;
#pragma unroll
    for (int s = 0; s < C3_STAGES - 1; ++s) {
        if (s < nk) load_stage(s, s * C3_KC);
        cp_commit();
    }

    for (int kt = 0; kt < nk; ++kt) {
        cp_wait<C3_STAGES - 2>();
        __syncthreads();
        {
            const int nxt = kt + C3_STAGES - 1;
            if (nxt < nk) load_stage(nxt % C3_STAGES, nxt * C3_KC);
            cp_commit();
        }
        const float *ar = sm3 + (size_t)(kt % C3_STAGES) * C3_STAGE, *ai = ar + C3_A_PLANE, *br = ai + C3_A_PLANE,
                    *bi = br + C3_B_PLANE;
#pragma unroll
        for (int ks = 0; ks < C3_KC / 8; ++ks) {
            // B fragments (k = 8 ks + t [+4], n = wn*32 + 8 ni + g), split
            unsigned brh[4][2], brl[4][2], bih[4][2], bil[4][2];
#pragma unroll
            for (int ni = 0; ni < 4; ++ni) {
                const int o = (wn * 32 + ni * 8 + g) * C3_LDB + ks * 8 + t;
                split_tf32(br[o], brh[ni][0], brl[ni][0]);
                split_tf32(br[o + 4], brh[ni][1], brl[ni][1]);
                split_tf32(bi[o], bih[ni][0], bil[ni][0]);
                split_tf32(bi[o + 4], bih[ni][1], bil[ni][1]);
            }
#pragma unroll
            for (int mi = 0; mi < 2; ++mi) {
                // A fragments (m = wm*32 + 16 mi + g [+8], k = 8 ks + t [+4]), split; -Ai for the real part
                unsigned arh[4], arl[4], aih[4], ail[4], nih[4], nil[4];
                const int o = (ks * 8 + t) * C3_LDA + wm * 32 + mi * 16 + g;
                split_tf32(ar[o], arh[0], arl[0]);
                split_tf32(ar[o + 8], arh[1], arl[1]);
                split_tf32(ar[o + 4 * C3_LDA], arh[2], arl[2]);
                split_tf32(ar[o + 4 * C3_LDA + 8], arh[3], arl[3]);
                split_tf32(ai[o], aih[0], ail[0]);
                split_tf32(ai[o + 8], aih[1], ail[1]);
                split_tf32(ai[o + 4 * C3_LDA], aih[2], ail[2]);
                split_tf32(ai[o + 4 * C3_LDA + 8], aih[3], ail[3]);
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    nih[e] = aih[e] ^ 0x80000000u;
                    nil[e] = ail[e] ^ 0x80000000u;
                }
#pragma unroll
                for (int ni = 0; ni < 4; ++ni) {
                    mma3(cr[mi][ni], arh, arl, brh[ni], brl[ni]);
                    mma3(cr[mi][ni], nih, nil, bih[ni], bil[ni]);
                    mma3(ci[mi][ni], arh, arl, bih[ni], bil[ni]);
                    mma3(ci[mi][ni], aih, ail, brh[ni], brl[ni]);
                }
            }
        }
    }
    cp_wait<0>();
    __syncthreads();

    // epilogue: c[0] (row g, col 2t), c[1] (g, 2t+1), c[2] (g+8, 2t), c[3] (g+8, 2t+1) of each 16 x 8 tile
#pragma unroll
    for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const long row = m0 + wm * 32 + mi * 16 + g + (e >> 1) * 8;
                const long col = n0 + wn * 32 + ni * 8 + 2 * t + (e & 1);
                if (row < M && col < N) {
                    float vr = alpha * cr[mi][ni][e], vi = alpha * ci[mi][ni][e];
                    if (beta != 0.f) {
                        vr = fmaf(beta, Cre[col * ldc + row], vr);
                        vi = fmaf(beta, Cim[col * ldc + row], vi);
                    }
                    Cre[col * ldc + row] = vr;
                    Cim[col * ldc + row] = vi;
                }
            }
}

}  // namespace

// C <- beta*C + alpha*A*B on split-complex float planes, 3xTF32.  Plane base addresses 16-byte aligned, lda and ldb
// multiples of 4 floats (met by every caller in lu.cu).
int cgemm3(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C) {
    return cgemm3_batched(st, m, n, k, alpha, A, 0, B, 0, beta, C, 0, 1);
}

// nbatch independent products; operand b of batch i lives at view + i * stride (in elements of a plane)
int cgemm3_batched(cudaStream_t st, int m, int n, int k, double alpha, CView A, long strideA, CView B, long strideB, double beta,
                   CView C, long strideC, int nbatch) {
    if (m <= 0 || n <= 0 || nbatch <= 0) return 0;
    if (k <= 0 && beta == 1.0) return 0;
    if (((uintptr_t)A.re | (uintptr_t)A.im | (uintptr_t)B.re | (uintptr_t)B.im) & 15) return -6;
    if ((A.ld | B.ld | strideA | strideB) & 3) return -7;
    static SmemCfg cfg;
    HP_TRY(configure_smem(cfg, cgemm3_kernel, C3_SMEM));
    const bool prof = prof_enabled() && k > 0;
    if (prof) prof_begin(st, 8.0 * m * n * k * nbatch);
    HP_CUDA(launch_pdl(cgemm3_kernel, dim3(ceil_div(m, C3_BM) * ceil_div(n, C3_BN), nbatch), dim3(C3_NT), C3_SMEM, st, m, n, k,
                       (float)alpha, A.re, A.im, (long)A.ld, B.re, B.im, (long)B.ld, (float)beta, C.re, C.im, (long)C.ld, strideA,
                       strideB, strideC));
    if (prof) prof_end(st);
    HP_LAUNCHED();
    return 0;
}

}  // namespace hp

extern "C" int hprmat_cgemm_3xtf32(void *cuda_stream, int m, int n, int k, float alpha, const float *A_re, const float *A_im,
                                   int lda, const float *B_re, const float *B_im, int ldb, float beta, float *C_re,
                                   float *C_im, int ldc) {
    if (m < 0) return -2;
    if (n < 0) return -3;
    if (k < 0) return -4;
    if (lda < (m > 1 ? m : 1) || (lda & 3)) return -8;
    if (ldb < (k > 1 ? k : 1) || (ldb & 3)) return -11;
    if (ldc < (m > 1 ? m : 1)) return -15;
    using namespace hp;
    return cgemm3_any((cudaStream_t)cuda_stream, m, n, k, alpha, CView((float *)A_re, (float *)A_im, lda),
                      CView((float *)B_re, (float *)B_im, ldb), beta, CView(C_re, C_im, ldc));
}
