// raw_mixed.cu -- hprmat_zsolve in the mixed modes: a general dense complex128 system solved with complex64 factors plus
// FP64 iterative refinement (PAPER.md:147-151 Type 2, :192-230 Type 4 / hybrid: z2c conversion, single-precision LU and
// solves, FP64 residual r = b - M x, correction solve, x += d; :561 non-convergence is detected and reported).
//
// The raw entry cannot know the block structure, so instead of the K_d^-1 preconditioner of the structured path the
// matrix is equilibrated: S = D_r A D_c with power-of-two row and column scalings (exact in floating point) that bring
// every row and column maximum to [1, 2), then demoted to planar complex64 and factorised by the same LU (single-pass TF32
// trailing update).  Refinement converges while kappa(S) * 2^-11 < 1; beyond that the call returns
// HPRMAT_ENOTCONVERGED with the last iterate (the paper's breakdown behaviour, Fig. 5) and the caller has HPRMAT_FP64.
#include <algorithm>

#include "lu.cuh"
#include "precond.cuh"
#include "refine.cuh"
#include "structured.cuh"

namespace hp {

namespace {

__device__ __forceinline__ double pow2_recip(double mx) {
    // 2^-e with 2^e <= mx < 2^(e+1); 1 for a zero row/column
    if (!(mx > 0.0)) return 1.0;
    int e;
    frexp(mx, &e);  // mx = f * 2^e, f in [0.5, 1)
    return ldexp(1.0, 1 - e);
}

// rs[i] = 2^-e of max_j |a_ij| ; rsum[i] = sum_j |a_ij| (moduli as |re| + |im| for the max, true modulus for the sum)
__global__ void __launch_bounds__(256) row_stats_kernel(int n, const double2 *__restrict__ A, long lda, double *rs, double *rsum) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double mx = 0.0, sm = 0.0;
    for (int j = 0; j < n; ++j) {
        const double2 a = A[(long)j * lda + i];
        mx = fmax(mx, fabs(a.x) + fabs(a.y));
        sm += sqrt(a.x * a.x + a.y * a.y);
    }
    rs[i] = pow2_recip(mx);
    rsum[i] = sm;
}

// cs[j] = 2^-e of max_i rs_i |a_ij| ; one CTA per column
__global__ void __launch_bounds__(256) col_scale_kernel(int n, const double2 *__restrict__ A, long lda, const double *__restrict__ rs,
                                                        double *cs) {
    __shared__ double sh[8];
    const int j = blockIdx.x;
    double mx = 0.0;
    for (int i = threadIdx.x; i < n; i += 256) {
        const double2 a = A[(long)j * lda + i];
        mx = fmax(mx, rs[i] * (fabs(a.x) + fabs(a.y)));
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, off));
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = mx;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) mx = fmax(mx, sh[w]);
        cs[j] = pow2_recip(mx);
    }
}

// S <- (complex64) rs_i a_ij cs_j, planar
__global__ void __launch_bounds__(256) equil_demote_kernel(int n, const double2 *__restrict__ A, long lda,
                                                           const double *__restrict__ rs, const double *__restrict__ cs,
                                                           float *__restrict__ re, float *__restrict__ im, long ld) {
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    const double r = rs[i];
    const int j0 = blockIdx.y * 8;
#pragma unroll
    for (int e = 0; e < 8; ++e) {
        const int j = j0 + e;
        if (j >= n) break;
        const double s = r * cs[j];
        const double2 a = A[(long)j * lda + i];
        re[(long)j * ld + i] = (float)(a.x * s);
        im[(long)j * ld + i] = (float)(a.y * s);
    }
}

// D <- (complex64) rs_i z_iq
__global__ void __launch_bounds__(256) scale_demote_kernel(long rows, int cols, const double2 *__restrict__ Z, long ldz,
                                                           const double *__restrict__ rs, float *__restrict__ re,
                                                           float *__restrict__ im, long ld) {
    const long tot = rows * cols;
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < tot; idx += (long)gridDim.x * blockDim.x) {
        const long q = idx / rows, r = idx - q * rows;
        const double2 z = Z[q * ldz + r];
        re[q * ld + r] = (float)(z.x * rs[r]);
        im[q * ld + r] = (float)(z.y * rs[r]);
    }
}

// X <- (accumulate ? X : 0) + cs_i d_iq ; norms[0] = max|cs d|, norms[1] = max|X_new|
__global__ void __launch_bounds__(256) promote_scale_add_kernel(long rows, int cols, double2 *__restrict__ X, long ldx,
                                                                const float *__restrict__ re, const float *__restrict__ im,
                                                                long ld, const double *__restrict__ cs, int accumulate,
                                                                double *norms) {
    __shared__ double shred[16];
    double md = 0.0, mx = 0.0;
    const long tot = rows * cols;
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < tot; idx += (long)gridDim.x * blockDim.x) {
        const long q = idx / rows, r = idx - q * rows;
        const double dr = cs[r] * (double)re[q * ld + r], di = cs[r] * (double)im[q * ld + r];
        double2 x = accumulate ? X[q * ldx + r] : make_double2(0.0, 0.0);
        x.x += dr;
        x.y += di;
        X[q * ldx + r] = x;
        md = fmax(md, sqrt(dr * dr + di * di));
        mx = fmax(mx, sqrt(x.x * x.x + x.y * x.y));
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        md = fmax(md, __shfl_xor_sync(0xffffffffu, md, off));
        mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, off));
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { shred[warp] = md; shred[8 + warp] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { md = fmax(md, shred[w]); mx = fmax(mx, shred[8 + w]); }
        atomicMax(reinterpret_cast<unsigned long long *>(norms), (unsigned long long)__double_as_longlong(md));
        atomicMax(reinterpret_cast<unsigned long long *>(norms + 1), (unsigned long long)__double_as_longlong(mx));
    }
}

// out[0] = max_i v_i
__global__ void __launch_bounds__(256) vecmax_kernel(int n, const double *__restrict__ v, double *out) {
    __shared__ double sh[8];
    double mx = 0.0;
    for (int i = blockIdx.x * 256 + threadIdx.x; i < n; i += gridDim.x * 256) mx = fmax(mx, v[i]);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, off));
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = mx;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) mx = fmax(mx, sh[w]);
        atomicMax(reinterpret_cast<unsigned long long *>(out), (unsigned long long)__double_as_longlong(mx));
    }
}

struct MixedWork {
    LuWork<CView> wk;
    CView S, Bs;
    double *rs, *cs, *rsum, *scal;
    double2 *B0, *R;
    int *info;
    size_t carve(void *base, int n, int nrhs) {
        char *p = (char *)base;
        auto take = [&](size_t bytes) {
            char *q = p;
            p += round_up((long)bytes, 256);
            return q;
        };
        p += wk.carve(p, n);
        const long ld = round_up(std::max(n, 1), 32);
        float *sre = (float *)take(sizeof(float) * ld * n), *sim = (float *)take(sizeof(float) * ld * n);
        S = CView(sre, sim, ld);
        float *bre = (float *)take(sizeof(float) * ld * std::max(nrhs, 1)), *bim = (float *)take(sizeof(float) * ld * std::max(nrhs, 1));
        Bs = CView(bre, bim, ld);
        rs = (double *)take(sizeof(double) * n);
        cs = (double *)take(sizeof(double) * n);
        rsum = (double *)take(sizeof(double) * n);
        scal = (double *)take(sizeof(double) * 16);
        B0 = (double2 *)take(sizeof(double2) * (size_t)n * std::max(nrhs, 1));
        R = (double2 *)take(sizeof(double2) * (size_t)n * std::max(nrhs, 1));
        info = (int *)take(256);
        return (size_t)(p - (char *)base);
    }
};

}  // namespace

size_t raw_workspace_mixed(int n, int nrhs) {
    MixedWork w;
    return w.carve((void *)0, n, nrhs);
}

int zgemm(cudaStream_t st, int m, int n, int k, double alpha, const double2 *A, long lda, const double2 *B, long ldb,
          double beta, double2 *C, long ldc);

int zsolve_mixed(cudaStream_t st, int n, int nrhs, const double2 *A, long lda, double2 *B, long ldb, int *ipiv, bool refine,
                 int max_refine, double tol, void *workspace, hprmat_info *info) {
    MixedWork w;
    w.carve(workspace, n, nrhs);
    if (max_refine < 0) max_refine = 12;  // the contraction per step is ~ sqrt(n) 2^-11 kappa(S): a few 1e-3 at best
    if (!refine) max_refine = 0;
    if (!(tol > 0.0)) tol = 1e-12;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    for (auto &e : ev) HP_CUDA(cudaEventCreate(&e));
    auto cleanup = [&]() { for (auto &e : ev) cudaEventDestroy(e); };
    int status = HPRMAT_OK, steps = 0;
    double h[8] = {0};
    int hinfo = 0;
#define ZM_TRY(x) do { int r__ = (x); if (r__ != 0) { cleanup(); return r__; } } while (0)
#define ZM_CUDA(x) do { cudaError_t e__ = (x); if (e__ != cudaSuccess) { cleanup(); return hp::cuda_fail(e__, __FILE__, __LINE__); } } while (0)
    ZM_CUDA(cudaEventRecord(ev[0], st));
    // keep b for the residual (PAPER.md:200-216 convert_z2c happens in equil_demote_kernel, fused with the scaling)
    ZM_CUDA(cudaMemcpy2DAsync(w.B0, sizeof(double2) * n, B, sizeof(double2) * ldb, sizeof(double2) * n, nrhs, cudaMemcpyDeviceToDevice, st));
    row_stats_kernel<<<ceil_div(n, 256), 256, 0, st>>>(n, A, lda, w.rs, w.rsum);
    HP_LAUNCHED();
    col_scale_kernel<<<n, 256, 0, st>>>(n, A, lda, w.rs, w.cs);
    HP_LAUNCHED();
    const int grid = (int)std::min<long>(ceil_div((long)n * nrhs, 256), 148L * 8);
    int fp32_class = 0;
    // Attempt 0: single-pass TF32 trailing update (contraction ~ sqrt(n) 2^-11 kappa per refinement step).  If the
    // refinement does not converge with those factors, attempt 1 refactors with FP32-class products everywhere (3xTF32:
    // contraction ~ sqrt(n) 2^-23 kappa), the paper's domain kappa u_FP32 < 1 (Fig. 5).
    for (int attempt = 0; attempt < 2; ++attempt) {
        w.wk.accurate = attempt == 1;
        fp32_class = attempt;
        steps = 0;
        ZM_CUDA(cudaMemsetAsync(w.info, 0, sizeof(int), st));
        ZM_CUDA(cudaMemsetAsync(w.scal, 0, sizeof(double) * 16, st));
        equil_demote_kernel<<<dim3(ceil_div(n, 256), ceil_div(n, 8)), 256, 0, st>>>(n, A, lda, w.rs, w.cs, w.S.re, w.S.im, w.S.ld);
        HP_LAUNCHED();
        vecmax_kernel<<<std::min(ceil_div(n, 256), 148), 256, 0, st>>>(n, w.rsum, w.scal + 4);  // ||A||_inf
        HP_LAUNCHED();
        ZM_TRY(getrf<CView>(st, n, w.S, ipiv, w.info, w.wk));
        ZM_CUDA(cudaEventRecord(ev[1], st));
        scale_demote_kernel<<<grid, 256, 0, st>>>(n, nrhs, w.B0, n, w.rs, w.Bs.re, w.Bs.im, w.Bs.ld);
        HP_LAUNCHED();
        ZM_TRY(getrs<CView>(st, n, nrhs, w.S, w.Bs, w.wk));
        promote_scale_add_kernel<<<grid, 256, 0, st>>>(n, nrhs, B, ldb, w.Bs.re, w.Bs.im, w.Bs.ld, w.cs, 0, w.scal);
        HP_LAUNCHED();
        ZM_CUDA(cudaEventRecord(ev[2], st));
        ZM_CUDA(cudaMemcpyAsync(h, w.scal, sizeof(double) * 2, cudaMemcpyDeviceToHost, st));
        ZM_CUDA(cudaMemcpyAsync(&hinfo, w.info, sizeof(int), cudaMemcpyDeviceToHost, st));
        ZM_CUDA(cudaStreamSynchronize(st));
        if (hinfo != 0) {
            cleanup();
            if (info) { info->status = HPRMAT_ESINGULAR; info->pivot_index = hinfo; }
            return HPRMAT_ESINGULAR;
        }
        double dprev = h[1];
        status = max_refine > 0 ? HPRMAT_ENOTCONVERGED : HPRMAT_OK;
        for (int k = 0; k < max_refine; ++k) {
            // r = b - A x in FP64 on the DMMA tensor cores
            ZM_CUDA(cudaMemcpyAsync(w.R, w.B0, sizeof(double2) * (size_t)n * nrhs, cudaMemcpyDeviceToDevice, st));
            ZM_TRY(zgemm(st, n, nrhs, n, -1.0, A, lda, B, ldb, 1.0, w.R, n));
            scale_demote_kernel<<<grid, 256, 0, st>>>(n, nrhs, w.R, n, w.rs, w.Bs.re, w.Bs.im, w.Bs.ld);
            HP_LAUNCHED();
            ZM_TRY(getrs<CView>(st, n, nrhs, w.S, w.Bs, w.wk));
            ZM_CUDA(cudaMemsetAsync(w.scal, 0, sizeof(double) * 2, st));
            promote_scale_add_kernel<<<grid, 256, 0, st>>>(n, nrhs, B, ldb, w.Bs.re, w.Bs.im, w.Bs.ld, w.cs, 1, w.scal);
            HP_LAUNCHED();
            ++steps;
            ZM_CUDA(cudaMemcpyAsync(h, w.scal, sizeof(double) * 2, cudaMemcpyDeviceToHost, st));
            ZM_CUDA(cudaStreamSynchronize(st));
            const int v = refine_verdict(h[0], h[1], dprev, tol);
            dprev = h[0];
            if (v == REF_CONVERGED) { status = HPRMAT_OK; break; }
            if (v == REF_STAGNATED) {
                status = (h[0] <= 64.0 * 2.220446049250313e-16 * h[1]) ? HPRMAT_OK : HPRMAT_ENOTCONVERGED;
                break;
            }
        }
        if (status == HPRMAT_ENOTCONVERGED && max_refine > 0) {
            // A correction that stopped shrinking is the attainable accuracy when x already solves the system to working
            // precision: for an ill-conditioned matrix the forward error floor is kappa 2^-53, not 2^-53.  Accept the iterate
            // if its backward error meets the north-star's FP64 bound 50 n 2^-53 (n floored at 64 for tiny systems).
            ZM_CUDA(cudaMemcpyAsync(w.R, w.B0, sizeof(double2) * (size_t)n * nrhs, cudaMemcpyDeviceToDevice, st));
            ZM_TRY(zgemm(st, n, nrhs, n, -1.0, A, lda, B, ldb, 1.0, w.R, n));
            ZM_TRY(maxabs(st, n, nrhs, w.B0, n, w.scal + 6));
            ZM_TRY(backward_error(st, n, nrhs, w.R, n, B, ldb, w.scal + 4, w.scal + 6, w.scal + 5));
            ZM_CUDA(cudaMemcpyAsync(h + 5, w.scal + 5, sizeof(double), cudaMemcpyDeviceToHost, st));
            ZM_CUDA(cudaStreamSynchronize(st));
            if (h[5] <= 50.0 * std::max(n, 64) * 1.1102230246251565e-16) status = HPRMAT_OK;
        }
        if (status == HPRMAT_OK || max_refine == 0) break;
    }
    w.wk.accurate = false;
    ZM_CUDA(cudaEventRecord(ev[3], st));
    if (info) {
        // backward error of the returned x: r = b - A x once more
        ZM_CUDA(cudaMemcpyAsync(w.R, w.B0, sizeof(double2) * (size_t)n * nrhs, cudaMemcpyDeviceToDevice, st));
        ZM_TRY(zgemm(st, n, nrhs, n, -1.0, A, lda, B, ldb, 1.0, w.R, n));
        ZM_TRY(maxabs(st, n, nrhs, w.R, n, w.scal + 3));
        ZM_TRY(maxabs(st, n, nrhs, w.B0, n, w.scal + 6));
        ZM_TRY(backward_error(st, n, nrhs, w.R, n, B, ldb, w.scal + 4, w.scal + 6, w.scal + 5));
        ZM_CUDA(cudaMemcpyAsync(h, w.scal, sizeof(double) * 8, cudaMemcpyDeviceToHost, st));
        ZM_CUDA(cudaStreamSynchronize(st));
        float ms = 0.f;
        info->status = status;
        info->refine_steps = steps;
        info->reserved = fp32_class;  // 1: the single-pass TF32 factors did not converge, FP32-class (3xTF32) factors were used
        info->resid_max = h[3];
        info->backward_err = h[5];
        cudaEventElapsedTime(&ms, ev[0], ev[1]);
        info->ms_lu = ms;
        cudaEventElapsedTime(&ms, ev[1], ev[2]);
        info->ms_solve = ms;
        cudaEventElapsedTime(&ms, ev[2], ev[3]);
        info->ms_refine = ms;
        cudaEventElapsedTime(&ms, ev[0], ev[3]);
        info->ms_total = ms;
        info->lu_tflops = info->ms_lu > 0 ? (8.0 / 3.0) * (double)n * n * n / (info->ms_lu * 1e-3) * 1e-12 : 0.0;
    }
#undef ZM_TRY
#undef ZM_CUDA
    cleanup();
    return status;
}

}  // namespace hp
