// ctx.cu -- the structured entries of the C ABI: hprmat_setup / mesh / solve / solve_host / get_x / get_matrix / destroy.
// Host side only sequences kernels on the context's stream; every arithmetic step of the path runs on the GPU.
//
// Setup (once per context, host, long double): Gauss-Legendre mesh on (0,a), surface values f_i(a)
// (the q2(r_i) of PAPER.md:85,133) and the kinetic + Bloch table T.  The paper only names these
// ("Lagrange-Legendre basis", refs [2],[3]); the closed forms are the standard ones of the Lagrange-mesh method
// regularised by r (reading R1):
//   x_i zeros of P_nb(2x-1), ascending;  f_i(a) = (-1)^(nb+i) / sqrt(a x_i (1-x_i)),  i = 1..nb
//   T_ii = [(4 nb^2 + 4 nb + 3) x_i (1-x_i) - 6 x_i + 1] / [3 a^2 x_i^2 (1-x_i)^2]
//   T_ij = (-1)^(i+j) / [a^2 sqrt(x_i x_j (1-x_i)(1-x_j))]
//          * [nb^2 + nb + 1 + (x_i + x_j - 2 x_i x_j)/(x_i - x_j)^2 - 1/(1-x_i) - 1/(1-x_j)]
#include <math.h>

#include <vector>

#include "lu.cuh"
#include "precond.cuh"
#include "refine.cuh"
#include "structured.cuh"

using namespace hp;

struct hprmat_ctx {
    int nch = 0, nb = 0, n = 0, max_mode = 0;
    double a = 0, h2m = 0;
    cudaStream_t st = nullptr;
    std::vector<double> r, fa;  // host copies for hprmat_mesh
    // device
    double *d_hT = nullptr, *d_dg0 = nullptr, *d_ethr = nullptr, *d_fa = nullptr;
    double2 *d_C = nullptr;                                   // N x N complex128 (FP64 mode)
    double2 *d_X = nullptr, *d_Rr = nullptr, *d_Rlo = nullptr;  // N x nch each
    double2 *d_V = nullptr, *d_R = nullptr;                   // staging for hprmat_solve_host
    void *d_work = nullptr;                                   // LU workspace
    int *d_ipiv = nullptr, *d_info = nullptr;
    double *d_scal = nullptr;                                 // small device scalars (norms, maxima)
    double *h_scal = nullptr;                                 // pinned mirror
    int *h_info = nullptr;                                    // pinned
    LuWork<ZView> wz;
    // mixed modes: split-complex64 system S = K_d^-1 (C - E I), its right-hand sides, the FP64 block inverses
    float *d_Sre = nullptr, *d_Sim = nullptr, *d_Bre = nullptr, *d_Bim = nullptr;
    double2 *d_Kinv = nullptr;
    void *d_workc = nullptr;
    long ldS = 0;
    LuWork<CView> wc;
    cudaEvent_t ev[8] = {};
    bool have_x = false;
    StructTables tab;
};

namespace {

typedef long double ld;

// P_n(t) and P_{n-1}(t) by the three-term recurrence
void legendre_pair(int n, ld t, ld &pn, ld &pm) {
    ld a = 1.0L, b = t;
    if (n == 0) { pn = 1.0L; pm = 0.0L; return; }
    for (int k = 1; k < n; ++k) {
        const ld c = ((2.0L * k + 1.0L) * t * b - (ld)k * a) / (ld)(k + 1);
        a = b;
        b = c;
    }
    pn = b;
    pm = a;
}

// zeros of P_n(2x-1) on (0,1), ascending, in long double; the upper half is found by Newton, the lower half mirrored
void shifted_legendre_zeros(int n, std::vector<ld> &x) {
    x.assign(n, 0.0L);
    const ld pi = acosl(-1.0L);
    for (int k = 0; k < (n + 1) / 2; ++k) {
        ld t = cosl(pi * (4.0L * (k + 1) - 1.0L) / (4.0L * n + 2.0L));  // k-th zero from the right end
        for (int it = 0; it < 60; ++it) {
            ld pn, pm;
            legendre_pair(n, t, pn, pm);
            const ld dp = (ld)n * (t * pn - pm) / (t * t - 1.0L);
            const ld dt = pn / dp;
            t -= dt;
            if (fabsl(dt) < 4e-20L) break;
        }
        if ((n & 1) && k == n / 2) t = 0.0L;
        x[n - 1 - k] = 0.5L * (1.0L + t);
        x[k] = 0.5L * (1.0L - t);
    }
}

int free_ctx(hprmat_ctx *c) {
    if (!c) return 0;
    cudaFree(c->d_hT); cudaFree(c->d_dg0); cudaFree(c->d_ethr); cudaFree(c->d_fa);
    cudaFree(c->d_C); cudaFree(c->d_X); cudaFree(c->d_Rr); cudaFree(c->d_Rlo); cudaFree(c->d_V); cudaFree(c->d_R);
    cudaFree(c->d_Sre); cudaFree(c->d_Sim); cudaFree(c->d_Bre); cudaFree(c->d_Bim); cudaFree(c->d_Kinv); cudaFree(c->d_workc);
    cudaFree(c->d_work); cudaFree(c->d_ipiv); cudaFree(c->d_info); cudaFree(c->d_scal);
    if (c->h_scal) cudaFreeHost(c->h_scal);
    if (c->h_info) cudaFreeHost(c->h_info);
    for (auto &e : c->ev)
        if (e) cudaEventDestroy(e);
    delete c;
    return 0;
}

#define HP_ALLOC(ptr, bytes)                                                  \
    do {                                                                      \
        cudaError_t e__ = cudaMalloc((void **)&(ptr), (bytes));               \
        if (e__ == cudaErrorMemoryAllocation) { cudaGetLastError(); free_ctx(c); return HPRMAT_ENOMEM; } \
        if (e__ != cudaSuccess) { free_ctx(c); return hp::cuda_fail(e__, __FILE__, __LINE__); }           \
    } while (0)

float ev_ms(cudaEvent_t a, cudaEvent_t b) {
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    return ms;
}

}  // namespace

extern "C" int hprmat_setup(hprmat_ctx **out, int nch, int nbasis, double a, double h2m, const int *lval,
                            const double *ethr, int max_mode, void *cuda_stream) {
    if (!out) return -1;
    *out = nullptr;
    if (nch < 1) return -2;
    if (nbasis < 2) return -3;
    if (!(a > 0.0)) return -4;
    if (!(h2m > 0.0)) return -5;
    if (!lval) return -6;
    if (!ethr) return -7;
    if ((long)nch * nbasis > 2000000000L / 16) return -2;
    const int all = (1 << HPRMAT_FP64) | (1 << HPRMAT_MIXED) | (1 << HPRMAT_MIXED_REFINE);
    if (max_mode == 0) max_mode = all;
    if (max_mode & ~all) return -8;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        snprintf(hp::g_cuda_err, sizeof(hp::g_cuda_err), "no CUDA device (there is no CPU fallback)");
        return HPRMAT_ECUDA;
    }
    hprmat_ctx *c = new hprmat_ctx;
    c->nch = nch; c->nb = nbasis; c->n = nch * nbasis; c->a = a; c->h2m = h2m; c->max_mode = max_mode;
    c->st = (cudaStream_t)cuda_stream;
    const int nb = nbasis;
    const long N = c->n;

    // ---- host tables (long double -> double, each value rounded once)
    std::vector<ld> xl;
    shifted_legendre_zeros(nb, xl);
    std::vector<double> x(nb), hT((size_t)nb * nb), dg0((size_t)N);
    c->r.resize(nb);
    c->fa.resize(nb);
    for (int i = 0; i < nb; ++i) {
        x[i] = (double)xl[i];
        c->r[i] = (double)((ld)a * xl[i]);
        const ld sgn = ((nb + i + 1) & 1) ? -1.0L : 1.0L;
        c->fa[i] = (double)(sgn / sqrtl((ld)a * xl[i] * (1.0L - xl[i])));
    }
    const ld n_ = nb, a2 = (ld)a * (ld)a;
    for (int j = 0; j < nb; ++j)
        for (int i = 0; i < nb; ++i) {
            const ld xi = x[i], xj = x[j];
            ld t;
            if (i == j) {
                const ld w = xi * (1.0L - xi);
                t = ((4.0L * n_ * n_ + 4.0L * n_ + 3.0L) * w - 6.0L * xi + 1.0L) / (3.0L * a2 * w * w);
            } else {
                const ld sg = ((i + j) & 1) ? -1.0L : 1.0L;
                const ld dx = xi - xj;
                t = sg / (a2 * sqrtl(xi * xj * (1.0L - xi) * (1.0L - xj))) *
                    (n_ * n_ + n_ + 1.0L + (xi + xj - 2.0L * xi * xj) / (dx * dx) - 1.0L / (1.0L - xi) - 1.0L / (1.0L - xj));
            }
            const double td = (double)t;
            hT[(size_t)j * nb + i] = h2m * td;  // the matrix entry: one FP64 product
        }
    for (int ch = 0; ch < nch; ++ch)
        for (int i = 0; i < nb; ++i) {
            const double l = lval[ch];
            const double cf = h2m * l * (l + 1) / (c->r[i] * c->r[i]);
            dg0[(size_t)ch * nb + i] = hT[(size_t)i * nb + i] + cf;
        }

    // ---- device buffers
    HP_ALLOC(c->d_hT, sizeof(double) * nb * nb);
    HP_ALLOC(c->d_dg0, sizeof(double) * N);
    HP_ALLOC(c->d_ethr, sizeof(double) * nch);
    HP_ALLOC(c->d_fa, sizeof(double) * nb);
    if (max_mode & (1 << HPRMAT_FP64)) {
        HP_ALLOC(c->d_C, sizeof(double2) * N * N);
        const size_t wb = LuWork<ZView>::bytes((int)N);
        HP_ALLOC(c->d_work, wb);
        c->wz.carve(c->d_work, (int)N);
        HP_ALLOC(c->d_Kinv, sizeof(double2) * (size_t)nch * nb * nb);
    }
    if (max_mode & ((1 << HPRMAT_MIXED) | (1 << HPRMAT_MIXED_REFINE))) {
        c->ldS = round_up(N, 32);
        HP_ALLOC(c->d_Sre, sizeof(float) * c->ldS * N);
        HP_ALLOC(c->d_Sim, sizeof(float) * c->ldS * N);
        HP_ALLOC(c->d_Bre, sizeof(float) * c->ldS * nch);
        HP_ALLOC(c->d_Bim, sizeof(float) * c->ldS * nch);
        if (!c->d_Kinv) HP_ALLOC(c->d_Kinv, sizeof(double2) * (size_t)nch * nb * nb);
        const size_t wb = LuWork<CView>::bytes((int)N);
        HP_ALLOC(c->d_workc, wb);
        if (cudaMemsetAsync(c->d_workc, 0, wb, c->st) != cudaSuccess) { free_ctx(c); return HPRMAT_ECUDA; }
        c->wc.carve(c->d_workc, (int)N);
        c->wc.speculate = true;  // S = I + K_d^-1 V: the diagonal is the partial-pivoting choice; verified per panel (panel.cu)
    }
    HP_ALLOC(c->d_X, sizeof(double2) * N * nch);
    HP_ALLOC(c->d_Rr, sizeof(double2) * N * nch);
    HP_ALLOC(c->d_Rlo, sizeof(double2) * N * nch);
    HP_ALLOC(c->d_V, sizeof(double2) * (size_t)nb * nch * nch);
    HP_ALLOC(c->d_R, sizeof(double2) * (size_t)nch * nch);
    HP_ALLOC(c->d_ipiv, sizeof(int) * N);
    HP_ALLOC(c->d_info, sizeof(int) * 4);
    HP_ALLOC(c->d_scal, sizeof(double) * 16);
    if (cudaMallocHost((void **)&c->h_scal, sizeof(double) * 16) != cudaSuccess ||
        cudaMallocHost((void **)&c->h_info, sizeof(int) * 4) != cudaSuccess) {
        cudaGetLastError();
        free_ctx(c);
        return HPRMAT_ENOMEM;
    }
    for (auto &e : c->ev)
        if (cudaEventCreate(&e) != cudaSuccess) { free_ctx(c); return HPRMAT_ECUDA; }
    cudaError_t e1 = cudaMemcpyAsync(c->d_hT, hT.data(), sizeof(double) * nb * nb, cudaMemcpyHostToDevice, c->st);
    cudaError_t e2 = cudaMemcpyAsync(c->d_dg0, dg0.data(), sizeof(double) * N, cudaMemcpyHostToDevice, c->st);
    cudaError_t e3 = cudaMemcpyAsync(c->d_ethr, ethr, sizeof(double) * nch, cudaMemcpyHostToDevice, c->st);
    cudaError_t e4 = cudaMemcpyAsync(c->d_fa, c->fa.data(), sizeof(double) * nb, cudaMemcpyHostToDevice, c->st);
    cudaError_t e5 = cudaStreamSynchronize(c->st);  // the host vectors go out of scope
    for (cudaError_t e : {e1, e2, e3, e4, e5})
        if (e != cudaSuccess) { free_ctx(c); return hp::cuda_fail(e, __FILE__, __LINE__); }
    c->tab.nch = nch; c->tab.nb = nb; c->tab.a = a; c->tab.h2m = h2m;
    c->tab.hT = c->d_hT; c->tab.dg0 = c->d_dg0; c->tab.ethr = c->d_ethr; c->tab.fa = c->d_fa;
    *out = c;
    return HPRMAT_OK;
}

extern "C" int hprmat_mesh(const hprmat_ctx *ctx, double *r, double *fa) {
    if (!ctx) return -1;
    for (int i = 0; i < ctx->nb; ++i) {
        if (r) r[i] = ctx->r[i];
        if (fa) fa[i] = ctx->fa[i];
    }
    return HPRMAT_OK;
}

extern "C" int hprmat_destroy(hprmat_ctx *ctx) {
    if (ctx) cudaStreamSynchronize(ctx->st);
    return free_ctx(ctx);
}

extern "C" int hprmat_get_matrix(hprmat_ctx *ctx, double energy, const void *V, void *C) {
    if (!ctx) return -1;
    if (!V) return -3;
    if (!C) return -4;
    return assemble_z(ctx->st, ctx->tab, energy, (const double2 *)V, (double2 *)C, ctx->n);
}

extern "C" int hprmat_get_x(const hprmat_ctx *ctx, void *X) {
    if (!ctx) return -1;
    if (!X) return -2;
    if (!ctx->have_x) return -1;
    HP_CUDA(cudaMemcpyAsync(X, ctx->d_X, sizeof(double2) * (size_t)ctx->n * ctx->nch, cudaMemcpyDeviceToDevice, ctx->st));
    return HPRMAT_OK;
}

namespace {

int solve_fp64(hprmat_ctx *c, double energy, const double2 *V, int max_refine, double tol, double2 *R, hprmat_info *info) {
    cudaStream_t st = c->st;
    const int N = c->n, nch = c->nch;
    const bool timed = info != nullptr;
    ZView A(c->d_C, N), X(c->d_X, N), D(c->d_Rr, N);
    if (max_refine < 0) max_refine = 2;
    if (!(tol > 0.0)) tol = 1e-13;
    int status = HPRMAT_OK, steps = 0;
    double rmax = 0.0;

    if (timed) HP_CUDA(cudaEventRecord(c->ev[0], st));
    HP_TRY(assemble_z(st, c->tab, energy, V, c->d_C, N));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[1], st));
    HP_CUDA(cudaMemsetAsync(c->d_info, 0, sizeof(int), st));
    HP_TRY(getrf<ZView>(st, N, A, c->d_ipiv, c->d_info, c->wz));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[2], st));
    if (timed) {
        HP_CUDA(cudaMemcpyAsync(c->h_info, c->d_info, sizeof(int), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        if (c->h_info[0] != 0) {
            info->status = HPRMAT_ESINGULAR;
            info->pivot_index = c->h_info[0];
            return HPRMAT_ESINGULAR;
        }
    }
    HP_TRY(build_rhs(st, c->tab, c->d_X, N));
    HP_TRY(getrs<ZView>(st, N, nch, A, X, c->wz));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[3], st));
    double dprev = 0.0;
    if (timed && max_refine > 0) {
        HP_TRY(maxabs(st, N, nch, c->d_X, N, c->d_scal + 2));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 2, c->d_scal + 2, sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        dprev = c->h_scal[2];
    }
    for (int k = 0; k < max_refine; ++k) {
        HP_TRY(structured_residual(st, c->tab, energy, V, nch, nullptr, 0, c->d_X, N, c->d_Rr, c->d_Rlo, N, c->d_scal + 3));
        HP_TRY(getrs<ZView>(st, N, nch, A, D, c->wz));
        HP_TRY(axpy_norm(st, N, nch, c->d_X, N, c->d_Rr, N, c->d_scal));
        ++steps;
        if (timed) {
            HP_CUDA(cudaMemcpyAsync(c->h_scal, c->d_scal, 4 * sizeof(double), cudaMemcpyDeviceToHost, st));
            HP_CUDA(cudaStreamSynchronize(st));
            const double dn = c->h_scal[0], xn = c->h_scal[1];
            rmax = c->h_scal[3];
            const int v = refine_verdict(dn, xn, dprev, tol);
            dprev = dn;
            if (v != REF_CONTINUE) break;  // FP64 mode: a stagnated correction is at the rounding floor, not a failure
        }
    }
    if (timed) HP_CUDA(cudaEventRecord(c->ev[4], st));
    HP_TRY(contract(st, c->tab, c->d_X, N, R));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[5], st));
    c->have_x = true;
    if (timed) {
        // backward error of the returned X (PAPER.md:139 accuracy reference; definition in DESIGN.md reading R8)
        HP_TRY(structured_residual(st, c->tab, energy, V, nch, nullptr, 0, c->d_X, N, c->d_Rr, c->d_Rlo, N, c->d_scal + 3));
        HP_TRY(structured_anorm(st, c->tab, energy, V, c->d_scal + 4));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 3, c->d_scal + 3, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        double bn = 0.0;
        for (double f : c->fa) bn = std::max(bn, fabs(f));
        HP_TRY(backward_error(st, N, nch, c->d_Rr, N, c->d_X, N, c->h_scal[4], bn, c->d_scal + 5));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 5, c->d_scal + 5, sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        info->status = status;
        info->refine_steps = steps;
        info->pivot_index = 0;
        info->resid_max = c->h_scal[3];
        info->backward_err = c->h_scal[5];
        info->ms_assemble = ev_ms(c->ev[0], c->ev[1]);
        info->ms_lu = ev_ms(c->ev[1], c->ev[2]);
        info->ms_solve = ev_ms(c->ev[2], c->ev[3]);
        info->ms_refine = ev_ms(c->ev[3], c->ev[4]);
        info->ms_contract = ev_ms(c->ev[4], c->ev[5]);
        info->ms_total = ev_ms(c->ev[0], c->ev[5]);
        info->lu_tflops = info->ms_lu > 0 ? (8.0 / 3.0) * (double)N * N * N / (info->ms_lu * 1e-3) * 1e-12 : 0.0;
        (void)rmax;
    }
    return status;
}

// FP64 mode, preconditioned form (the default; hprmat_fp64_algo): the FP64 LU is applied to S = K_d^-1 (C - E I), the matrix
// of the paper's Type 3 (Eqs. 7-9), instead of C - E I itself.  Same N x N complex LU with partial pivoting and the same
// 8N^3/3 flops, but S = I + (coupling-sized entries): the pivots partial pivoting selects are the diagonal ones, which the
// speculative panel (panel.cu) verifies column by column -- the sequential pivot search across all SMs (N dependent
// exchanges, ~0.1 s at N = 25600) disappears, and with kappa(S) = O(1) the first solve is already at the rounding floor.
// The residual of the refinement and the reported backward error are those of the ORIGINAL system (C - E I) X = B.
constexpr int PRECOND_UNUSABLE = -1000;  // internal: the synchronised call falls back to the LU of C - E I

int solve_fp64_precond(hprmat_ctx *c, double energy, const double2 *V, int max_refine, double tol, double2 *R,
                       hprmat_info *info) {
    cudaStream_t st = c->st;
    const int N = c->n, nch = c->nch, nb = c->nb;
    const bool timed = info != nullptr;
    ZView S(c->d_C, N), X(c->d_X, N), D(c->d_Rlo, N);
    if (max_refine < 0) max_refine = 2;
    if (!(tol > 0.0)) tol = 1e-13;
    int steps = 0;

    if (timed) HP_CUDA(cudaEventRecord(c->ev[0], st));
    HP_CUDA(cudaMemsetAsync(c->d_info, 0, 2 * sizeof(int), st));
    HP_TRY(precond_invert(st, c->tab, energy, V, c->d_Kinv, c->d_info + 1));
    HP_TRY(precond_assemble_z(st, c->tab, c->d_Kinv, V, S));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[1], st));
    c->wz.speculate = true;
    const int rc_lu = getrf<ZView>(st, N, S, c->d_ipiv, c->d_info, c->wz);
    c->wz.speculate = false;
    HP_TRY(rc_lu);
    if (timed) HP_CUDA(cudaEventRecord(c->ev[2], st));
    if (timed) {
        HP_CUDA(cudaMemcpyAsync(c->h_info, c->d_info, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        if (c->h_info[0] != 0 || c->h_info[1] != 0) return PRECOND_UNUSABLE;  // e.g. E on a pole of an uncoupled channel
    }
    HP_TRY(precond_rhs_z(st, c->tab, c->d_Kinv, X));
    HP_TRY(getrs<ZView>(st, N, nch, S, X, c->wz));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[3], st));
    double dprev = 0.0;
    if (timed && max_refine > 0) {
        HP_TRY(maxabs(st, N, nch, c->d_X, N, c->d_scal + 2));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 2, c->d_scal + 2, sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        dprev = c->h_scal[2];
    }
    for (int k = 0; k < max_refine; ++k) {
        HP_TRY(structured_residual(st, c->tab, energy, V, nch, nullptr, 0, c->d_X, N, c->d_Rr, c->d_Rlo, N, c->d_scal + 3));
        // z = K_d^-1 r (one nb x nb by nb x nch product per channel), d = S^-1 z
        HP_TRY(zgemm_batched(st, nb, nch, nb, 1.0, c->d_Kinv, nb, (long)nb * nb, c->d_Rr, N, nb, 0.0, c->d_Rlo, N, nb, nch));
        HP_TRY(getrs<ZView>(st, N, nch, S, D, c->wz));
        HP_TRY(axpy_norm(st, N, nch, c->d_X, N, c->d_Rlo, N, c->d_scal));
        ++steps;
        if (timed) {
            HP_CUDA(cudaMemcpyAsync(c->h_scal, c->d_scal, 4 * sizeof(double), cudaMemcpyDeviceToHost, st));
            HP_CUDA(cudaStreamSynchronize(st));
            const double dn = c->h_scal[0], xn = c->h_scal[1];
            const int v = refine_verdict(dn, xn, dprev, tol);
            dprev = dn;
            if (v != REF_CONTINUE) {
                // FP64 mode: a stagnated correction is at the rounding floor, not a failure -- unless it is large: then the
                // preconditioner is ill-conditioned at this energy (near a pole of an uncoupled channel)
                if (!(dn <= 1e-9 * xn)) return PRECOND_UNUSABLE;
                break;
            }
        }
    }
    if (timed) HP_CUDA(cudaEventRecord(c->ev[4], st));
    HP_TRY(contract(st, c->tab, c->d_X, N, R));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[5], st));
    c->have_x = true;
    if (timed) {
        HP_TRY(structured_residual(st, c->tab, energy, V, nch, nullptr, 0, c->d_X, N, c->d_Rr, c->d_Rlo, N, c->d_scal + 3));
        HP_TRY(structured_anorm(st, c->tab, energy, V, c->d_scal + 4));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 3, c->d_scal + 3, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        double bn = 0.0;
        for (double f : c->fa) bn = std::max(bn, fabs(f));
        HP_TRY(backward_error(st, N, nch, c->d_Rr, N, c->d_X, N, c->h_scal[4], bn, c->d_scal + 5));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 5, c->d_scal + 5, sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        if (!(c->h_scal[5] <= 50.0 * N * 1.1102230246251565e-16)) return PRECOND_UNUSABLE;
        info->status = HPRMAT_OK;
        info->refine_steps = steps;
        info->pivot_index = 0;
        info->resid_max = c->h_scal[3];
        info->backward_err = c->h_scal[5];
        info->ms_assemble = ev_ms(c->ev[0], c->ev[1]);
        info->ms_lu = ev_ms(c->ev[1], c->ev[2]);
        info->ms_solve = ev_ms(c->ev[2], c->ev[3]);
        info->ms_refine = ev_ms(c->ev[3], c->ev[4]);
        info->ms_contract = ev_ms(c->ev[4], c->ev[5]);
        info->ms_total = ev_ms(c->ev[0], c->ev[5]);
        info->lu_tflops = info->ms_lu > 0 ? (8.0 / 3.0) * (double)N * N * N / (info->ms_lu * 1e-3) * 1e-12 : 0.0;
    }
    return HPRMAT_OK;
}

// Mixed modes (PAPER.md:147-151 Type 2, :192-230 Type 4; preconditioned per reading R10):
//   Kinv = K_d^-1 (FP64) -> S = K_d^-1 (C - E I) in split complex64 -> P L U = S (TF32 tensor-core trailing update)
//   -> X0 = S^-1 (K_d^-1 B)  [HPRMAT_MIXED stops here]
//   -> repeat: r = B - (C - E I) X (FP64, double-double, matrix-free); z = K_d^-1 r (FP64); d = S^-1 z (complex64
//      factors); X += d; until the correction is below tol or stagnates.
int solve_mixed(hprmat_ctx *c, double energy, const double2 *V, bool refine, int max_refine, double tol, double2 *R,
                hprmat_info *info) {
    cudaStream_t st = c->st;
    const int N = c->n, nch = c->nch, nb = c->nb;
    const bool timed = info != nullptr;
    CView S(c->d_Sre, c->d_Sim, c->ldS), Bs(c->d_Bre, c->d_Bim, c->ldS);
    if (max_refine < 0) max_refine = 5;
    if (!refine) max_refine = 0;
    if (!(tol > 0.0)) tol = 1e-12;  // estimated relative error left in X; the north-star asks 1e-10 of R
    int status = HPRMAT_OK, steps = 0;

    if (timed) HP_CUDA(cudaEventRecord(c->ev[0], st));
    HP_CUDA(cudaMemsetAsync(c->d_info, 0, 2 * sizeof(int), st));
    HP_TRY(precond_invert(st, c->tab, energy, V, c->d_Kinv, c->d_info + 1));
    HP_TRY(precond_assemble(st, c->tab, c->d_Kinv, V, S));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[1], st));
    HP_TRY(getrf<CView>(st, N, S, c->d_ipiv, c->d_info, c->wc));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[2], st));
    if (timed) {
        HP_CUDA(cudaMemcpyAsync(c->h_info, c->d_info, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        if (c->h_info[0] != 0 || c->h_info[1] != 0) {
            info->status = HPRMAT_ESINGULAR;
            info->pivot_index = c->h_info[0] ? c->h_info[0] : c->h_info[1];
            return HPRMAT_ESINGULAR;
        }
    }
    HP_TRY(precond_rhs(st, c->tab, c->d_Kinv, Bs));
    HP_TRY(getrs<CView>(st, N, nch, S, Bs, c->wc));
    HP_TRY(promote_add(st, N, nch, c->d_X, N, Bs, false, c->d_scal));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[3], st));
    double dprev = 0.0;
    if (max_refine > 0) {
        HP_CUDA(cudaMemcpyAsync(c->h_scal, c->d_scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        dprev = c->h_scal[1];
        status = HPRMAT_ENOTCONVERGED;
    }
    for (int k = 0; k < max_refine; ++k) {
        HP_TRY(structured_residual(st, c->tab, energy, V, nch, nullptr, 0, c->d_X, N, c->d_Rr, c->d_Rlo, N, c->d_scal + 3));
        // z = K_d^-1 r: one nb x nb by nb x nch product per channel (FP64 tensor cores), into Rlo
        HP_TRY(zgemm_batched(st, nb, nch, nb, 1.0, c->d_Kinv, nb, (long)nb * nb, c->d_Rr, N, nb, 0.0, c->d_Rlo, N, nb, nch));
        HP_TRY(demote(st, N, nch, c->d_Rlo, N, Bs));
        HP_TRY(getrs<CView>(st, N, nch, S, Bs, c->wc));
        HP_TRY(promote_add(st, N, nch, c->d_X, N, Bs, true, c->d_scal));
        ++steps;
        HP_CUDA(cudaMemcpyAsync(c->h_scal, c->d_scal, 4 * sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        const double dn = c->h_scal[0], xn = c->h_scal[1];
        const int v = refine_verdict(dn, xn, dprev, tol);
        dprev = dn;
        if (v == REF_CONVERGED) { status = HPRMAT_OK; break; }
        if (v == REF_STAGNATED) {
            // a correction at the FP64 rounding floor of X is convergence, not failure
            status = (dn <= 64.0 * 2.220446049250313e-16 * xn) ? HPRMAT_OK : HPRMAT_ENOTCONVERGED;
            break;
        }
    }
    if (timed) HP_CUDA(cudaEventRecord(c->ev[4], st));
    HP_TRY(contract(st, c->tab, c->d_X, N, R));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[5], st));
    c->have_x = true;
    if (timed) {
        HP_TRY(structured_residual(st, c->tab, energy, V, nch, nullptr, 0, c->d_X, N, c->d_Rr, c->d_Rlo, N, c->d_scal + 3));
        HP_TRY(structured_anorm(st, c->tab, energy, V, c->d_scal + 4));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 3, c->d_scal + 3, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        double bn = 0.0;
        for (double f : c->fa) bn = std::max(bn, fabs(f));
        HP_TRY(backward_error(st, N, nch, c->d_Rr, N, c->d_X, N, c->h_scal[4], bn, c->d_scal + 5));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 5, c->d_scal + 5, sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        info->status = status;
        info->refine_steps = steps;
        info->pivot_index = 0;
        info->resid_max = c->h_scal[3];
        info->backward_err = c->h_scal[5];
        info->ms_assemble = ev_ms(c->ev[0], c->ev[1]);
        info->ms_lu = ev_ms(c->ev[1], c->ev[2]);
        info->ms_solve = ev_ms(c->ev[2], c->ev[3]);
        info->ms_refine = ev_ms(c->ev[3], c->ev[4]);
        info->ms_contract = ev_ms(c->ev[4], c->ev[5]);
        info->ms_total = ev_ms(c->ev[0], c->ev[5]);
        info->lu_tflops = info->ms_lu > 0 ? (8.0 / 3.0) * (double)N * N * N / (info->ms_lu * 1e-3) * 1e-12 : 0.0;
    }
    return status;
}

}  // namespace

static int g_fp64_algo = 2;  // hprmat_fp64_algo

// Non-local potentials: the same path with a dense potential matrix W.
// Residual of the refinement: B - (K + W) X = [structured residual with V = 0, double-double] - W X, the product W X on the
// FP64 tensor cores (the LU has overwritten C, W is the caller's and intact), i.e. a working-precision residual as in
// LAPACK's refinement: it restores the backward error, it does not add digits beyond kappa * 2^-53.
static int nonlocal_residual(hprmat_ctx *c, double energy, const double2 *W, long ldw, double *rmax_dev) {
    cudaStream_t st = c->st;
    const int N = c->n, nch = c->nch;
    HP_TRY(structured_residual(st, c->tab, energy, c->d_V, nch, nullptr, 0, c->d_X, N, c->d_Rr, c->d_Rlo, N, nullptr));
    HP_TRY(gemm(st, N, nch, N, -1.0, ZView((double2 *)W, ldw), ZView(c->d_X, N), 1.0, ZView(c->d_Rr, N)));
    if (rmax_dev) HP_TRY(maxabs(st, N, nch, c->d_Rr, N, rmax_dev));
    return 0;
}

static int solve_nonlocal_fp64(hprmat_ctx *c, double energy, const double2 *W, long ldw, int max_refine, double tol,
                               double2 *R, hprmat_info *info) {
    cudaStream_t st = c->st;
    const int N = c->n, nch = c->nch;
    const bool timed = info != nullptr;
    ZView A(c->d_C, N), X(c->d_X, N), D(c->d_Rr, N);
    if (max_refine < 0) max_refine = 2;
    if (!(tol > 0.0)) tol = 1e-13;
    int steps = 0;

    if (timed) HP_CUDA(cudaEventRecord(c->ev[0], st));
    HP_CUDA(cudaMemsetAsync(c->d_V, 0, sizeof(double2) * (size_t)c->nb * nch * nch, st));  // "no local potential"
    HP_TRY(assemble_nonlocal(st, c->tab, energy, W, ldw, c->d_C, N));
    if (timed) HP_TRY(nonlocal_anorm(st, c->tab, energy, W, ldw, (double *)c->d_Rlo, c->d_scal + 4));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[1], st));
    HP_CUDA(cudaMemsetAsync(c->d_info, 0, sizeof(int), st));
    HP_TRY(getrf<ZView>(st, N, A, c->d_ipiv, c->d_info, c->wz));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[2], st));
    if (timed) {
        HP_CUDA(cudaMemcpyAsync(c->h_info, c->d_info, sizeof(int), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        if (c->h_info[0] != 0) {
            info->status = HPRMAT_ESINGULAR;
            info->pivot_index = c->h_info[0];
            return HPRMAT_ESINGULAR;
        }
    }
    HP_TRY(build_rhs(st, c->tab, c->d_X, N));
    HP_TRY(getrs<ZView>(st, N, nch, A, X, c->wz));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[3], st));
    double dprev = 0.0;
    if (timed && max_refine > 0) {
        HP_TRY(maxabs(st, N, nch, c->d_X, N, c->d_scal + 2));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 2, c->d_scal + 2, sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        dprev = c->h_scal[2];
    }
    for (int k = 0; k < max_refine; ++k) {
        HP_TRY(nonlocal_residual(c, energy, W, ldw, nullptr));
        HP_TRY(getrs<ZView>(st, N, nch, A, D, c->wz));
        HP_TRY(axpy_norm(st, N, nch, c->d_X, N, c->d_Rr, N, c->d_scal));
        ++steps;
        if (timed) {
            HP_CUDA(cudaMemcpyAsync(c->h_scal, c->d_scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
            HP_CUDA(cudaStreamSynchronize(st));
            const double dn = c->h_scal[0], xn = c->h_scal[1];
            const int v = refine_verdict(dn, xn, dprev, tol);
            dprev = dn;
            if (v != REF_CONTINUE) break;
        }
    }
    if (timed) HP_CUDA(cudaEventRecord(c->ev[4], st));
    HP_TRY(contract(st, c->tab, c->d_X, N, R));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[5], st));
    c->have_x = true;
    if (timed) {
        HP_TRY(nonlocal_residual(c, energy, W, ldw, c->d_scal + 3));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 3, c->d_scal + 3, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        double bn = 0.0;
        for (double f : c->fa) bn = std::max(bn, fabs(f));
        HP_TRY(backward_error(st, N, nch, c->d_Rr, N, c->d_X, N, c->h_scal[4], bn, c->d_scal + 5));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 5, c->d_scal + 5, sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        info->status = HPRMAT_OK;
        info->refine_steps = steps;
        info->pivot_index = 0;
        info->resid_max = c->h_scal[3];
        info->backward_err = c->h_scal[5];
        info->ms_assemble = ev_ms(c->ev[0], c->ev[1]);
        info->ms_lu = ev_ms(c->ev[1], c->ev[2]);
        info->ms_solve = ev_ms(c->ev[2], c->ev[3]);
        info->ms_refine = ev_ms(c->ev[3], c->ev[4]);
        info->ms_contract = ev_ms(c->ev[4], c->ev[5]);
        info->ms_total = ev_ms(c->ev[0], c->ev[5]);
        info->lu_tflops = info->ms_lu > 0 ? (8.0 / 3.0) * (double)N * N * N / (info->ms_lu * 1e-3) * 1e-12 : 0.0;
    }
    return HPRMAT_OK;
}

// FP64 mode with non-local potentials, preconditioned form (hprmat_fp64_algo = 2): S = K_d^-1 (K + W) in FP64 with the full
// diagonal blocks K_c + W_cc inverted; block row c of S is one batched DMMA product Kinv_c x (block row c of W), the diagonal
// blocks are then overwritten by the identity.  Verified diagonal pivots as in solve_fp64_precond.
__global__ void __launch_bounds__(256) set_diag_blocks_identity_kernel(int nch, int nb, double2 *__restrict__ S, long ld) {
    const long tot = (long)nch * nb * nb;
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < tot; idx += (long)gridDim.x * blockDim.x) {
        const int c = (int)(idx / ((long)nb * nb));
        const int rem = (int)(idx - (long)c * nb * nb);
        const int i = rem % nb, j = rem / nb;
        S[((long)c * nb + j) * ld + (long)c * nb + i] = make_double2(i == j ? 1.0 : 0.0, 0.0);
    }
}

static int solve_nonlocal_fp64_precond(hprmat_ctx *c, double energy, const double2 *W, long ldw, int max_refine, double tol,
                                       double2 *R, hprmat_info *info) {
    cudaStream_t st = c->st;
    const int N = c->n, nch = c->nch, nb = c->nb;
    const bool timed = info != nullptr;
    ZView S(c->d_C, N), X(c->d_X, N), D(c->d_Rlo, N);
    if (max_refine < 0) max_refine = 2;
    if (!(tol > 0.0)) tol = 1e-13;
    int steps = 0;

    if (timed) HP_CUDA(cudaEventRecord(c->ev[0], st));
    HP_CUDA(cudaMemsetAsync(c->d_V, 0, sizeof(double2) * (size_t)nb * nch * nch, st));  // "no local potential"
    HP_CUDA(cudaMemsetAsync(c->d_info, 0, 2 * sizeof(int), st));
    HP_TRY(precond_invert(st, c->tab, energy, c->d_V, c->d_Kinv, c->d_info + 1, W, ldw));
    HP_TRY(zgemm_batched(st, nb, N, nb, 1.0, c->d_Kinv, nb, (long)nb * nb, W, ldw, nb, 0.0, c->d_C, N, nb, nch));
    {
        const long tot = (long)nch * nb * nb;
        set_diag_blocks_identity_kernel<<<(int)std::min<long>((tot + 255) / 256, 148 * 8), 256, 0, st>>>(nch, nb, c->d_C, N);
        HP_LAUNCHED();
    }
    if (timed) HP_TRY(nonlocal_anorm(st, c->tab, energy, W, ldw, (double *)c->d_Rlo, c->d_scal + 4));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[1], st));
    c->wz.speculate = true;
    const int rc_lu = getrf<ZView>(st, N, S, c->d_ipiv, c->d_info, c->wz);
    c->wz.speculate = false;
    HP_TRY(rc_lu);
    if (timed) HP_CUDA(cudaEventRecord(c->ev[2], st));
    if (timed) {
        HP_CUDA(cudaMemcpyAsync(c->h_info, c->d_info, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        if (c->h_info[0] != 0 || c->h_info[1] != 0) return PRECOND_UNUSABLE;
    }
    HP_TRY(precond_rhs_z(st, c->tab, c->d_Kinv, X));
    HP_TRY(getrs<ZView>(st, N, nch, S, X, c->wz));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[3], st));
    double dprev = 0.0;
    if (timed && max_refine > 0) {
        HP_TRY(maxabs(st, N, nch, c->d_X, N, c->d_scal + 2));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 2, c->d_scal + 2, sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        dprev = c->h_scal[2];
    }
    for (int k = 0; k < max_refine; ++k) {
        HP_TRY(nonlocal_residual(c, energy, W, ldw, nullptr));
        HP_TRY(zgemm_batched(st, nb, nch, nb, 1.0, c->d_Kinv, nb, (long)nb * nb, c->d_Rr, N, nb, 0.0, c->d_Rlo, N, nb, nch));
        HP_TRY(getrs<ZView>(st, N, nch, S, D, c->wz));
        HP_TRY(axpy_norm(st, N, nch, c->d_X, N, c->d_Rlo, N, c->d_scal));
        ++steps;
        if (timed) {
            HP_CUDA(cudaMemcpyAsync(c->h_scal, c->d_scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
            HP_CUDA(cudaStreamSynchronize(st));
            const double dn = c->h_scal[0], xn = c->h_scal[1];
            const int v = refine_verdict(dn, xn, dprev, tol);
            dprev = dn;
            if (v != REF_CONTINUE) {
                if (!(dn <= 1e-9 * xn)) return PRECOND_UNUSABLE;
                break;
            }
        }
    }
    if (timed) HP_CUDA(cudaEventRecord(c->ev[4], st));
    HP_TRY(contract(st, c->tab, c->d_X, N, R));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[5], st));
    c->have_x = true;
    if (timed) {
        HP_TRY(nonlocal_residual(c, energy, W, ldw, c->d_scal + 3));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 3, c->d_scal + 3, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        double bn = 0.0;
        for (double f : c->fa) bn = std::max(bn, fabs(f));
        HP_TRY(backward_error(st, N, nch, c->d_Rr, N, c->d_X, N, c->h_scal[4], bn, c->d_scal + 5));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 5, c->d_scal + 5, sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        if (!(c->h_scal[5] <= 50.0 * N * 1.1102230246251565e-16)) return PRECOND_UNUSABLE;
        info->status = HPRMAT_OK;
        info->refine_steps = steps;
        info->pivot_index = 0;
        info->resid_max = c->h_scal[3];
        info->backward_err = c->h_scal[5];
        info->ms_assemble = ev_ms(c->ev[0], c->ev[1]);
        info->ms_lu = ev_ms(c->ev[1], c->ev[2]);
        info->ms_solve = ev_ms(c->ev[2], c->ev[3]);
        info->ms_refine = ev_ms(c->ev[3], c->ev[4]);
        info->ms_contract = ev_ms(c->ev[4], c->ev[5]);
        info->ms_total = ev_ms(c->ev[0], c->ev[5]);
        info->lu_tflops = info->ms_lu > 0 ? (8.0 / 3.0) * (double)N * N * N / (info->ms_lu * 1e-3) * 1e-12 : 0.0;
    }
    return HPRMAT_OK;
}

// Mixed modes with non-local potentials: the block-diagonal preconditioner uses the full diagonal blocks K_c + W_cc, S has
// full off-diagonal blocks Kinv_c W_cc'; the rest is solve_mixed with the working-precision dense residual.
static int solve_nonlocal_mixed(hprmat_ctx *c, double energy, const double2 *W, long ldw, bool refine, int max_refine,
                                double tol, double2 *R, hprmat_info *info) {
    cudaStream_t st = c->st;
    const int N = c->n, nch = c->nch, nb = c->nb;
    const bool timed = info != nullptr;
    CView S(c->d_Sre, c->d_Sim, c->ldS), Bs(c->d_Bre, c->d_Bim, c->ldS);
    if (max_refine < 0) max_refine = 5;
    if (!refine) max_refine = 0;
    if (!(tol > 0.0)) tol = 1e-12;
    int status = HPRMAT_OK, steps = 0;

    if (timed) HP_CUDA(cudaEventRecord(c->ev[0], st));
    HP_CUDA(cudaMemsetAsync(c->d_V, 0, sizeof(double2) * (size_t)nb * nch * nch, st));  // "no local potential"
    HP_CUDA(cudaMemsetAsync(c->d_info, 0, 2 * sizeof(int), st));
    HP_TRY(precond_invert(st, c->tab, energy, c->d_V, c->d_Kinv, c->d_info + 1, W, ldw));
    HP_TRY(precond_assemble_nonlocal(st, c->tab, c->d_Kinv, W, ldw, S, c->d_Rlo, N));
    if (timed) HP_TRY(nonlocal_anorm(st, c->tab, energy, W, ldw, (double *)c->d_Rlo, c->d_scal + 4));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[1], st));
    HP_TRY(getrf<CView>(st, N, S, c->d_ipiv, c->d_info, c->wc));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[2], st));
    if (timed) {
        HP_CUDA(cudaMemcpyAsync(c->h_info, c->d_info, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        if (c->h_info[0] != 0 || c->h_info[1] != 0) {
            info->status = HPRMAT_ESINGULAR;
            info->pivot_index = c->h_info[0] ? c->h_info[0] : c->h_info[1];
            return HPRMAT_ESINGULAR;
        }
    }
    HP_TRY(precond_rhs(st, c->tab, c->d_Kinv, Bs));
    HP_TRY(getrs<CView>(st, N, nch, S, Bs, c->wc));
    HP_TRY(promote_add(st, N, nch, c->d_X, N, Bs, false, c->d_scal));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[3], st));
    double dprev = 0.0;
    if (max_refine > 0) {
        HP_CUDA(cudaMemcpyAsync(c->h_scal, c->d_scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        dprev = c->h_scal[1];
        status = HPRMAT_ENOTCONVERGED;
    }
    for (int k = 0; k < max_refine; ++k) {
        HP_TRY(nonlocal_residual(c, energy, W, ldw, nullptr));
        HP_TRY(zgemm_batched(st, nb, nch, nb, 1.0, c->d_Kinv, nb, (long)nb * nb, c->d_Rr, N, nb, 0.0, c->d_Rlo, N, nb, nch));
        HP_TRY(demote(st, N, nch, c->d_Rlo, N, Bs));
        HP_TRY(getrs<CView>(st, N, nch, S, Bs, c->wc));
        HP_TRY(promote_add(st, N, nch, c->d_X, N, Bs, true, c->d_scal));
        ++steps;
        HP_CUDA(cudaMemcpyAsync(c->h_scal, c->d_scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        const double dn = c->h_scal[0], xn = c->h_scal[1];
        const int v = refine_verdict(dn, xn, dprev, tol);
        dprev = dn;
        if (v == REF_CONVERGED) { status = HPRMAT_OK; break; }
        if (v == REF_STAGNATED) {
            status = (dn <= 64.0 * 2.220446049250313e-16 * xn) ? HPRMAT_OK : HPRMAT_ENOTCONVERGED;
            break;
        }
    }
    if (timed) HP_CUDA(cudaEventRecord(c->ev[4], st));
    HP_TRY(contract(st, c->tab, c->d_X, N, R));
    if (timed) HP_CUDA(cudaEventRecord(c->ev[5], st));
    c->have_x = true;
    if (timed) {
        HP_TRY(nonlocal_residual(c, energy, W, ldw, c->d_scal + 3));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 3, c->d_scal + 3, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        double bn = 0.0;
        for (double f : c->fa) bn = std::max(bn, fabs(f));
        HP_TRY(backward_error(st, N, nch, c->d_Rr, N, c->d_X, N, c->h_scal[4], bn, c->d_scal + 5));
        HP_CUDA(cudaMemcpyAsync(c->h_scal + 5, c->d_scal + 5, sizeof(double), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        info->status = status;
        info->refine_steps = steps;
        info->pivot_index = 0;
        info->resid_max = c->h_scal[3];
        info->backward_err = c->h_scal[5];
        info->ms_assemble = ev_ms(c->ev[0], c->ev[1]);
        info->ms_lu = ev_ms(c->ev[1], c->ev[2]);
        info->ms_solve = ev_ms(c->ev[2], c->ev[3]);
        info->ms_refine = ev_ms(c->ev[3], c->ev[4]);
        info->ms_contract = ev_ms(c->ev[4], c->ev[5]);
        info->ms_total = ev_ms(c->ev[0], c->ev[5]);
        info->lu_tflops = info->ms_lu > 0 ? (8.0 / 3.0) * (double)N * N * N / (info->ms_lu * 1e-3) * 1e-12 : 0.0;
    }
    return status;
}

extern "C" int hprmat_solve_nonlocal(hprmat_ctx *ctx, double energy, const void *W, long ldw, int mode, int max_refine,
                                     double tol, void *R, hprmat_info *info) {
    if (!ctx) return -1;
    if (!W) return -3;
    if (ldw < ctx->n) return -4;
    if (mode != HPRMAT_FP64 && mode != HPRMAT_MIXED && mode != HPRMAT_MIXED_REFINE) return -5;
    if (!(ctx->max_mode & (1 << mode))) return -5;
    if (!R) return -8;
    if (info) {
        *info = hprmat_info();
        info->backward_err = -1.0;
    }
    if (mode == HPRMAT_FP64 && g_fp64_algo == 2) {
        int rc2 = solve_nonlocal_fp64_precond(ctx, energy, (const double2 *)W, ldw, max_refine, tol, (double2 *)R, info);
        if (rc2 == PRECOND_UNUSABLE) {  // synchronised calls only
            *info = hprmat_info();
            info->backward_err = -1.0;
            rc2 = solve_nonlocal_fp64(ctx, energy, (const double2 *)W, ldw, max_refine, tol, (double2 *)R, info);
        }
        if (info) info->status = rc2;
        return rc2;
    }
    const int rc = mode == HPRMAT_FP64
                       ? solve_nonlocal_fp64(ctx, energy, (const double2 *)W, ldw, max_refine, tol, (double2 *)R, info)
                       : solve_nonlocal_mixed(ctx, energy, (const double2 *)W, ldw, mode == HPRMAT_MIXED_REFINE, max_refine, tol,
                                              (double2 *)R, info);
    if (info) info->status = rc;
    return rc;
}

extern "C" int hprmat_fp64_algo(int algo) {
    if (algo == 1 || algo == 2) g_fp64_algo = algo;
    return g_fp64_algo;
}

extern "C" int hprmat_solve(hprmat_ctx *ctx, double energy, const void *V, int mode, int max_refine, double tol, void *R,
                            hprmat_info *info) {
    if (!ctx) return -1;
    if (!V) return -3;
    if (mode != HPRMAT_FP64 && mode != HPRMAT_MIXED && mode != HPRMAT_MIXED_REFINE) return -4;
    if (!(ctx->max_mode & (1 << mode))) return -4;
    if (!R) return -7;
    if (info) {
        *info = hprmat_info();
        info->backward_err = -1.0;
    }
    int rc;
    if (mode == HPRMAT_FP64) {
        rc = g_fp64_algo == 2 ? solve_fp64_precond(ctx, energy, (const double2 *)V, max_refine, tol, (double2 *)R, info)
                              : solve_fp64(ctx, energy, (const double2 *)V, max_refine, tol, (double2 *)R, info);
        if (rc == PRECOND_UNUSABLE) {  // only reachable from a synchronised call (info != NULL)
            *info = hprmat_info();
            info->backward_err = -1.0;
            rc = solve_fp64(ctx, energy, (const double2 *)V, max_refine, tol, (double2 *)R, info);
        }
    } else {
        rc = solve_mixed(ctx, energy, (const double2 *)V, mode == HPRMAT_MIXED_REFINE, max_refine, tol, (double2 *)R, info);
    }
    if (info) info->status = rc;
    return rc;
}

extern "C" int hprmat_solve_host(hprmat_ctx *ctx, double energy, const void *V_host, int mode, int max_refine, double tol,
                                 void *R_host, hprmat_info *info) {
    if (!ctx) return -1;
    if (!V_host) return -3;
    if (!R_host) return -7;
    const size_t vb = sizeof(double2) * (size_t)ctx->nb * ctx->nch * ctx->nch, rb = sizeof(double2) * (size_t)ctx->nch * ctx->nch;
    HP_CUDA(cudaMemcpyAsync(ctx->d_V, V_host, vb, cudaMemcpyHostToDevice, ctx->st));
    const int rc = hprmat_solve(ctx, energy, ctx->d_V, mode, max_refine, tol, ctx->d_R, info);
    if (rc != HPRMAT_OK && rc != HPRMAT_ENOTCONVERGED) return rc;
    HP_CUDA(cudaMemcpyAsync(R_host, ctx->d_R, rb, cudaMemcpyDeviceToHost, ctx->st));
    HP_CUDA(cudaStreamSynchronize(ctx->st));
    return rc;
}
