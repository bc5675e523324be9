// ctx.cu -- the structured entries of the C ABI: hprmat_setup / mesh / solve / solve_nonlocal / solve_host / get_x /
// get_matrix / last_status / set_option / destroy.
// Host side only sequences kernels on the context's stream; every arithmetic step of the path runs on the GPU, including
// the stopping rule of the refinement (refine_verdict_kernel): a synchronised call reads the device status once, at the end.
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

#include <algorithm>
#include <vector>

#include "lu.cuh"
#include "precond.cuh"
#include "refine.cuh"
#include "structured.cuh"
#include "../../include/hprmat_profile.h"

using namespace hp;

struct hprmat_ctx {
    int nch = 0, nb = 0, n = 0, max_mode = 0;
    double a = 0, h2m = 0;
    cudaStream_t st = nullptr;
    std::vector<double> r, fa;  // host copies for hprmat_mesh
    // sub-interval contexts (hprmat_setup_sector): (a_lo, a), surface values at the LEFT end (fa holds the right end's)
    bool sector = false;
    double a_lo = 0;
    std::vector<double> fa_left;
    double *d_fa_left = nullptr;
    double2 *d_Rsec = nullptr;  // scratch: one nch x nch block
    // device
    double *d_hT = nullptr, *d_dg0 = nullptr, *d_ethr = nullptr, *d_fa = nullptr;
    double *d_KTinv = nullptr, *d_cf = nullptr, *d_g = nullptr;  // Type 3: (h2m T)^-1, centrifugal terms, (h2m T)^-1 q2
    double2 *d_C = nullptr;                                   // N x N complex128 (FP64 mode)
    double2 *d_X = nullptr, *d_Rr = nullptr, *d_Rlo = nullptr;  // N x nch each
    double2 *d_V = nullptr, *d_R = nullptr;                   // staging for hprmat_solve_host
    double2 *d_Voff = nullptr, *d_Xp = nullptr, *d_Pp = nullptr;  // residual: V without its diagonal, point-major X, V X
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
    // per-context settings (0 = follow the process default), see hprmat_set_option
    int fp64_algo = 0, zgemm_algo = 0;
    // side stream of the factorisations of this context + its fork/join events
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    cudaStream_t la_stream[LuWork<ZView>::NLA] = {};   // look-ahead streams / events of the factorisations (lu.cuh)
    cudaEvent_t la_fork[LuWork<ZView>::NLA] = {}, la_join[LuWork<ZView>::NLA] = {};
    // refinement steps the last solve in each mode took: that many are enqueued before the single read-back of the next
    // solve (index: HPRMAT_FP64 .. HPRMAT_MIXED_REFINE)
    int plan_steps[5] = {0, 1, 0, 2, 0};
    // what the last solve was, for hprmat_last_status
    int last_fac = -1, last_mode = 0, last_max_refine = 0;
    bool last_valid = false, last_fallback = false;
    bool reuse_factor = false;  // the next run keeps the factors of the previous one (second right-hand-side set of a sector)
    // CUDA graphs of the factorisations and triangular solves (thousands of dependent launches that depend on nothing but
    // this context's buffers): captured once on an internal stream, replayed on the caller's stream
    struct GraphEntry {
        int kind;              // 0 = getrf, 1 = getrs
        int flags;             // factored matrix / pivoting variant / right-hand-side count
        const void *key;       // right-hand-side buffer (getrs)
        cudaGraphExec_t exec;  // nullptr: capture is not possible for this entry, run it eagerly
        long long launches;    // kernel launches one replay stands for
    };
    std::vector<GraphEntry> graphs;
    cudaStream_t cap = nullptr;  // capture stream
    int use_graphs = 1;
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
    cudaFree(c->d_KTinv); cudaFree(c->d_cf); cudaFree(c->d_g); cudaFree(c->d_fa_left); cudaFree(c->d_Rsec);
    cudaFree(c->d_hT); cudaFree(c->d_dg0); cudaFree(c->d_ethr); cudaFree(c->d_fa);
    cudaFree(c->d_Voff); cudaFree(c->d_Xp); cudaFree(c->d_Pp);
    cudaFree(c->d_C); cudaFree(c->d_X); cudaFree(c->d_Rr); cudaFree(c->d_Rlo); cudaFree(c->d_V); cudaFree(c->d_R);
    cudaFree(c->d_Sre); cudaFree(c->d_Sim); cudaFree(c->d_Bre); cudaFree(c->d_Bim); cudaFree(c->d_Kinv); cudaFree(c->d_workc);
    cudaFree(c->d_work); cudaFree(c->d_ipiv); cudaFree(c->d_info); cudaFree(c->d_scal);
    if (c->h_scal) cudaFreeHost(c->h_scal);
    if (c->h_info) cudaFreeHost(c->h_info);
    for (auto &e : c->ev)
        if (e) cudaEventDestroy(e);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->side) cudaStreamDestroy(c->side);
    for (int d = 0; d < LuWork<ZView>::NLA; ++d) {
        if (c->la_fork[d]) cudaEventDestroy(c->la_fork[d]);
        if (c->la_join[d]) cudaEventDestroy(c->la_join[d]);
        if (c->la_stream[d]) cudaStreamDestroy(c->la_stream[d]);
    }
    for (auto &g : c->graphs)
        if (g.exec) cudaGraphExecDestroy(g.exec);
    if (c->cap) cudaStreamDestroy(c->cap);
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

// a_lo == 0: the interval (0, a) with the mesh regularised by r (hprmat_setup).  a_lo > 0: the sub-interval (a_lo, a) of a
// propagation (hprmat_setup_sector): plain Lagrange-Legendre mesh, Bloch operators at both ends.
static int setup_impl(hprmat_ctx **out, int nch, int nbasis, double a_lo, double a, double h2m, const int *lval,
                      const double *ethr, int max_mode, void *cuda_stream) {
    if (!out) return -1;
    *out = nullptr;
    if (nch < 1) return -2;
    if (nbasis < 2) return -3;
    if (!(a > 0.0) || !(a_lo >= 0.0) || !(a > a_lo)) return -4;
    if (!(h2m > 0.0)) return -5;
    if (!lval) return -6;
    if (!ethr) return -7;
    if ((long)nch * nbasis > 2000000000L / 16) return -2;
    const int all = (1 << HPRMAT_FP64) | (1 << HPRMAT_MIXED) | (1 << HPRMAT_MIXED_REFINE) | (1 << HPRMAT_TYPE3);
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
    c->sector = a_lo > 0.0;
    c->a_lo = a_lo;
    if (c->sector) {
        // Sub-interval (a_lo, a), h = a - a_lo (reading R16): Lagrange functions f_i(r) = l_i(x) / sqrt(h lam_i),
        // x = (r - a_lo)/h, l_i the Lagrange polynomials of the nb Gauss-Legendre nodes, lam_i the weights on (0,1).  With
        // the Bloch operator at BOTH ends,  <f_i| -d2/dr2 + L(a) - L(a_lo) |f_j> = int f_i' f_j' dr
        //   = (1/h^2) sum_k lam_k l_i'(x_k) l_j'(x_k) / sqrt(lam_i lam_j)    (Gauss quadrature, exact: degree 2 nb - 4),
        // l_i'(x_k) from the barycentric weights w_i = 1 / prod_{m != i} (x_i - x_m):
        //   l_i'(x_k) = (w_i / w_k) / (x_k - x_i)  (k != i),   l_k'(x_k) = - sum_{i != k} l_i'(x_k).
        const ld h = (ld)a - (ld)a_lo;
        std::vector<ld> lam(nb), wb(nb), D((size_t)nb * nb);
        for (int i = 0; i < nb; ++i) {
            const ld t = 2.0L * xl[i] - 1.0L;
            ld pn, pm;
            legendre_pair(nb, t, pn, pm);
            const ld dp = (ld)nb * (t * pn - pm) / (t * t - 1.0L);
            lam[i] = 1.0L / ((1.0L - t * t) * dp * dp);
            ld prod = 1.0L;
            for (int m = 0; m < nb; ++m)
                if (m != i) prod *= (xl[i] - xl[m]);
            wb[i] = 1.0L / prod;
        }
        for (int k = 0; k < nb; ++k) {
            ld sum = 0.0L;
            for (int i = 0; i < nb; ++i)
                if (i != k) {
                    D[(size_t)k * nb + i] = (wb[i] / wb[k]) / (xl[k] - xl[i]);  // l_i'(x_k)
                    sum += D[(size_t)k * nb + i];
                }
            D[(size_t)k * nb + k] = -sum;
        }
        c->fa_left.resize(nb);
        for (int i = 0; i < nb; ++i) {
            x[i] = (double)xl[i];
            c->r[i] = (double)((ld)a_lo + h * xl[i]);
            ld l0 = wb[i], l1 = wb[i];  // l_i(0), l_i(1)
            for (int m = 0; m < nb; ++m)
                if (m != i) { l0 *= (0.0L - xl[m]); l1 *= (1.0L - xl[m]); }
            c->fa_left[i] = (double)(l0 / sqrtl(h * lam[i]));
            c->fa[i] = (double)(l1 / sqrtl(h * lam[i]));  // right end: the surface the R-matrix is propagated to
        }
        for (int j = 0; j < nb; ++j)
            for (int i = 0; i < nb; ++i) {
                ld t = 0.0L;
                for (int k = 0; k < nb; ++k) t += lam[k] * D[(size_t)k * nb + i] * D[(size_t)k * nb + j];
                t /= (h * h * sqrtl(lam[i] * lam[j]));
                hT[(size_t)j * nb + i] = h2m * (double)t;
            }
    } else {
    for (int i = 0; i < nb; ++i) {
        x[i] = (double)xl[i];
        c->r[i] = (double)((ld)a * xl[i]);
        const ld sgn = ((nb + i + 1) & 1) ? -1.0L : 1.0L;
        c->fa[i] = (double)(sgn / sqrtl((ld)a * xl[i] * (1.0L - xl[i])));
    }
    }
    const ld n_ = nb, a2 = (ld)a * (ld)a;
    for (int j = 0; j < nb && !c->sector; ++j)
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

    // ---- Type 3: the kinetic block K = h2m T is real, shared by all channels and ENERGY-INDEPENDENT, so its
    //      inverse (step 1 of the paper's algorithm; Gauss-Jordan with partial pivoting in long double here), the
    //      transformed surface vector K^-1 q2 of Eq. (9) and the centrifugal terms are computed once per context
    std::vector<double> KTinv, cfv, gv;
    if (max_mode & (1 << HPRMAT_TYPE3)) {
        std::vector<ld> aug((size_t)nb * 2 * nb);
        for (int i = 0; i < nb; ++i)
            for (int j = 0; j < nb; ++j) {
                aug[(size_t)i * 2 * nb + j] = (ld)hT[(size_t)j * nb + i];
                aug[(size_t)i * 2 * nb + nb + j] = i == j ? 1.0L : 0.0L;
            }
        for (int k = 0; k < nb; ++k) {
            int piv = k;
            for (int i = k + 1; i < nb; ++i)
                if (fabsl(aug[(size_t)i * 2 * nb + k]) > fabsl(aug[(size_t)piv * 2 * nb + k])) piv = i;
            if (piv != k)
                for (int j = 0; j < 2 * nb; ++j) std::swap(aug[(size_t)k * 2 * nb + j], aug[(size_t)piv * 2 * nb + j]);
            const ld d = aug[(size_t)k * 2 * nb + k];
            if (d == 0.0L) { free_ctx(c); return -3; }  // cannot happen: T is positive definite
            for (int j = 0; j < 2 * nb; ++j) aug[(size_t)k * 2 * nb + j] /= d;
            for (int i = 0; i < nb; ++i) {
                if (i == k) continue;
                const ld f = aug[(size_t)i * 2 * nb + k];
                if (f == 0.0L) continue;
                for (int j = 0; j < 2 * nb; ++j) aug[(size_t)i * 2 * nb + j] -= f * aug[(size_t)k * 2 * nb + j];
            }
        }
        KTinv.resize((size_t)nb * nb);
        gv.assign(nb, 0.0);
        for (int i = 0; i < nb; ++i) {
            ld g = 0.0L;
            for (int j = 0; j < nb; ++j) {
                KTinv[(size_t)j * nb + i] = (double)aug[(size_t)i * 2 * nb + nb + j];
                g += aug[(size_t)i * 2 * nb + nb + j] * (ld)c->fa[j];
            }
            gv[i] = (double)g;
        }
        cfv.resize((size_t)N);
        for (int ch = 0; ch < nch; ++ch)
            for (int i = 0; i < nb; ++i) {
                const double l = lval[ch];
                cfv[(size_t)ch * nb + i] = h2m * l * (l + 1) / (c->r[i] * c->r[i]);
            }
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
    if (max_mode & ((1 << HPRMAT_MIXED) | (1 << HPRMAT_MIXED_REFINE) | (1 << HPRMAT_TYPE3))) {
        c->ldS = round_up(N, 32);
        HP_ALLOC(c->d_Sre, sizeof(float) * c->ldS * N);
        HP_ALLOC(c->d_Sim, sizeof(float) * c->ldS * N);
        HP_ALLOC(c->d_Bre, sizeof(float) * c->ldS * nch);
        HP_ALLOC(c->d_Bim, sizeof(float) * c->ldS * nch);
        if (!c->d_Kinv) HP_ALLOC(c->d_Kinv, sizeof(double2) * (size_t)nch * nb * nb);
        const size_t wb = LuWork<CView>::bytes((int)N, true);
        HP_ALLOC(c->d_workc, wb);
        if (cudaMemsetAsync(c->d_workc, 0, wb, c->st) != cudaSuccess) { free_ctx(c); return HPRMAT_ECUDA; }
        c->wc.carve(c->d_workc, (int)N, true);
        c->wc.speculate = true;  // S = I + K_d^-1 V: the diagonal is the partial-pivoting choice; verified (toplu.cu)
    }
    HP_ALLOC(c->d_X, sizeof(double2) * N * nch);
    HP_ALLOC(c->d_Rr, sizeof(double2) * N * nch);
    HP_ALLOC(c->d_Rlo, sizeof(double2) * N * nch);
    HP_ALLOC(c->d_V, sizeof(double2) * (size_t)nb * nch * nch);
    HP_ALLOC(c->d_Voff, sizeof(double2) * (size_t)nb * nch * nch);
    HP_ALLOC(c->d_Xp, sizeof(double2) * N * nch);
    HP_ALLOC(c->d_Pp, sizeof(double2) * N * nch);
    HP_ALLOC(c->d_R, sizeof(double2) * (size_t)nch * nch);
    HP_ALLOC(c->d_ipiv, sizeof(int) * N);
    HP_ALLOC(c->d_info, sizeof(int) * IN_NWORDS);
    HP_ALLOC(c->d_scal, sizeof(double) * SC_NWORDS);
    if (cudaMallocHost((void **)&c->h_scal, sizeof(double) * SC_NWORDS) != cudaSuccess ||
        cudaMallocHost((void **)&c->h_info, sizeof(int) * IN_NWORDS) != cudaSuccess) {
        cudaGetLastError();
        free_ctx(c);
        return HPRMAT_ENOMEM;
    }
    for (auto &e : c->ev)
        if (cudaEventCreate(&e) != cudaSuccess) { free_ctx(c); return HPRMAT_ECUDA; }
    if (cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&c->cap, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        free_ctx(c);
        return HPRMAT_ECUDA;
    }
    for (int d = 0; d < LuWork<ZView>::NLA; ++d) {
        if (cudaStreamCreateWithFlags(&c->la_stream[d], cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->la_fork[d], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->la_join[d], cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();
            free_ctx(c);
            return HPRMAT_ECUDA;
        }
        c->wz.la_stream[d] = c->wc.la_stream[d] = c->la_stream[d];
        c->wz.la_fork[d] = c->wc.la_fork[d] = c->la_fork[d];
        c->wz.la_join[d] = c->wc.la_join[d] = c->la_join[d];
    }
    for (LuWork<ZView> *w : {&c->wz}) { w->side = c->side; w->ev_fork = c->ev_fork; w->ev_join = c->ev_join; w->refuted = c->d_info + IN_REFUTED; }
    for (LuWork<CView> *w : {&c->wc}) { w->side = c->side; w->ev_fork = c->ev_fork; w->ev_join = c->ev_join; w->refuted = c->d_info + IN_REFUTED; }
    {   // ||B||_inf of the surface right-hand sides, read by the backward-error kernel from device memory
        double bn = 0.0;
        for (double f : c->fa) bn = std::max(bn, fabs(f));
        cudaError_t e0 = cudaMemsetAsync(c->d_scal, 0, sizeof(double) * SC_NWORDS, c->st);
        cudaError_t e1 = cudaMemcpyAsync(c->d_scal + SC_BNORM, &bn, sizeof(double), cudaMemcpyHostToDevice, c->st);
        cudaError_t e2 = cudaMemsetAsync(c->d_info, 0, sizeof(int) * IN_NWORDS, c->st);
        cudaError_t e3 = cudaStreamSynchronize(c->st);
        for (cudaError_t e : {e0, e1, e2, e3})
            if (e != cudaSuccess) { free_ctx(c); return hp::cuda_fail(e, __FILE__, __LINE__); }
    }
    cudaError_t e1 = cudaMemcpyAsync(c->d_hT, hT.data(), sizeof(double) * nb * nb, cudaMemcpyHostToDevice, c->st);
    cudaError_t e2 = cudaMemcpyAsync(c->d_dg0, dg0.data(), sizeof(double) * N, cudaMemcpyHostToDevice, c->st);
    cudaError_t e3 = cudaMemcpyAsync(c->d_ethr, ethr, sizeof(double) * nch, cudaMemcpyHostToDevice, c->st);
    cudaError_t e4 = cudaMemcpyAsync(c->d_fa, c->fa.data(), sizeof(double) * nb, cudaMemcpyHostToDevice, c->st);
    if (max_mode & (1 << HPRMAT_TYPE3)) {
        HP_ALLOC(c->d_KTinv, sizeof(double) * nb * nb);
        HP_ALLOC(c->d_cf, sizeof(double) * N);
        HP_ALLOC(c->d_g, sizeof(double) * nb);
        cudaError_t t1 = cudaMemcpyAsync(c->d_KTinv, KTinv.data(), sizeof(double) * nb * nb, cudaMemcpyHostToDevice, c->st);
        cudaError_t t2 = cudaMemcpyAsync(c->d_cf, cfv.data(), sizeof(double) * N, cudaMemcpyHostToDevice, c->st);
        cudaError_t t3 = cudaMemcpyAsync(c->d_g, gv.data(), sizeof(double) * nb, cudaMemcpyHostToDevice, c->st);
        for (cudaError_t e : {t1, t2, t3})
            if (e != cudaSuccess) { free_ctx(c); return hp::cuda_fail(e, __FILE__, __LINE__); }
    }
    cudaError_t e5 = cudaStreamSynchronize(c->st);  // the host vectors go out of scope
    for (cudaError_t e : {e1, e2, e3, e4, e5})
        if (e != cudaSuccess) { free_ctx(c); return hp::cuda_fail(e, __FILE__, __LINE__); }
    c->tab.nch = nch; c->tab.nb = nb; c->tab.a = c->sector ? 1.0 : a; c->tab.h2m = h2m;  // sector: no 1/a in the contraction
    if (c->sector) {
        HP_ALLOC(c->d_fa_left, sizeof(double) * nb);
        HP_ALLOC(c->d_Rsec, sizeof(double2) * (size_t)nch * nch);
        cudaError_t s1 = cudaMemcpy(c->d_fa_left, c->fa_left.data(), sizeof(double) * nb, cudaMemcpyHostToDevice);
        if (s1 != cudaSuccess) { free_ctx(c); return hp::cuda_fail(s1, __FILE__, __LINE__); }
    }
    c->tab.hT = c->d_hT; c->tab.dg0 = c->d_dg0; c->tab.ethr = c->d_ethr; c->tab.fa = c->d_fa;
    *out = c;
    return HPRMAT_OK;
}

extern "C" int hprmat_setup(hprmat_ctx **out, int nch, int nbasis, double a, double h2m, const int *lval,
                            const double *ethr, int max_mode, void *cuda_stream) {
    return setup_impl(out, nch, nbasis, 0.0, a, h2m, lval, ethr, max_mode, cuda_stream);
}

extern "C" int hprmat_setup_sector(hprmat_ctx **out, int nch, int nbasis, double a_lo, double a_hi, double h2m, const int *lval,
                                   const double *ethr, int max_mode, void *cuda_stream) {
    if (!(a_lo > 0.0)) return -4;
    if (!(a_hi > a_lo)) return -5;
    if (max_mode & (1 << HPRMAT_TYPE3)) return -9;  // Type 3 is printed for the single interval only
    if (max_mode == 0) max_mode = (1 << HPRMAT_FP64) | (1 << HPRMAT_MIXED) | (1 << HPRMAT_MIXED_REFINE);
    const int rc = setup_impl(out, nch, nbasis, a_lo, a_hi, h2m, lval, ethr, max_mode, cuda_stream);
    return rc == -4 ? -5 : rc == -5 ? -6 : rc == -6 ? -7 : rc == -7 ? -8 : rc == -8 ? -9 : rc;
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


// ======================================================================================================================
// One driver for every structured solve.  What varies:
//   the problem   local potentials V (mesh-diagonal couplings, Eq. 4) or a dense non-local potential matrix W (reading R15);
//   the factored matrix
//     FAC_C_Z   C - E I itself, FP64 LU with partial pivoting               (the paper's Type 1)
//     FAC_S_Z   S = K_d^-1 (C - E I) in FP64, verified diagonal pivots      (the matrix of the paper's Type 3, Eqs. 7-9)
//     FAC_S_C   S in planar complex64, TF32 tensor-core trailing update     (Types 2/4)
//     FAC_T3    the paper's Type 3 LITERALLY (Eqs. 7-9): point-major Schur matrix I + K^-1 V with the real, shared,
//               energy-independent kinetic block K; complex64 LU with partial pivoting and FP32-class (3xTF32) products
//               (kappa(S) ~ 1e5: single-pass TF32 would cost 1e-3 ... 1e-2 in R); no refinement
//   whether non-convergence of the refinement is an error (mixed+refine) or the rounding floor (FP64).
// Residual, stopping rule and reported backward error always refer to the ORIGINAL system (C - E I) X = B.
// ======================================================================================================================
namespace {

enum Fac { FAC_C_Z = 0, FAC_S_Z = 1, FAC_S_C = 2, FAC_T3 = 3 };
constexpr int UNUSABLE = -1000;  // internal: the verified-diagonal factorisation cannot be trusted here (refuted pivots,
                                 // singular diagonal block, ill-conditioned preconditioner): factor with pivoting instead

struct Problem {
    const double2 *V = nullptr;  // local: dev [nb][nch][nch]; non-local: the context's zeroed d_V ("no local potential")
    const double2 *W = nullptr;  // non-local: dev N x N, ld ldw
    long ldw = 0;
};

// ---- the device-side stopping rule --------------------------------------------------------------------------------------
__global__ void refine_begin_kernel(double *scal, int *info, int x0_word) {
    scal[SC_DPREV] = scal[x0_word];
    scal[SC_DN_LAST] = 0.0;
    scal[SC_XN_LAST] = scal[x0_word];
    info[IN_VERDICT] = REF_CONTINUE;
    info[IN_STEPS] = 0;
}
// after the (gated) update of step k: norms of the correction and of X are in scal[SC_DN], scal[SC_XN]
__global__ void refine_verdict_kernel(double *scal, int *info, double tol) {
    if (info[IN_VERDICT] != REF_CONTINUE) return;  // stopped earlier: this step did not touch X
    const double dn = scal[SC_DN], xn = scal[SC_XN];
    info[IN_VERDICT] = refine_verdict(dn, xn, scal[SC_DPREV], tol);
    info[IN_STEPS] += 1;
    scal[SC_DPREV] = dn;
    scal[SC_DN_LAST] = dn;
    scal[SC_XN_LAST] = xn;
}

// FP64 mode with non-local potentials, preconditioned form: block row c of S is one batched DMMA product Kinv_c x (block
// row c of W); the diagonal blocks are then overwritten by the identity.
__global__ void __launch_bounds__(256) set_diag_blocks_identity_kernel(int nch, int nb, double2 *__restrict__ S, long ld) {
    const long tot = (long)nch * nb * nb;
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < tot; idx += (long)gridDim.x * blockDim.x) {
        const int c = (int)(idx / ((long)nb * nb));
        const int rem = (int)(idx - (long)c * nb * nb);
        const int i = rem % nb, j = rem / nb;
        S[((long)c * nb + j) * ld + (long)c * nb + i] = make_double2(i == j ? 1.0 : 0.0, 0.0);
    }
}

// ---- CUDA-graph replay of a launch sequence that depends on the context's buffers only ---------------------------------
// enqueue(stream) issues the sequence.  First use: it is captured on the context's capture stream (the side stream joins the
// capture through its fork/join events) and instantiated; afterwards one cudaGraphLaunch on the caller's stream stands
// for it.  Anything that cannot be captured (or the per-launch timing of hprmat_profile, which needs real launches) runs
// eagerly on the caller's stream, as before.
template <class F> int replay(hprmat_ctx *c, int kind, int flags, const void *key, F &&enqueue) {
    if (!c->use_graphs || prof_enabled()) return enqueue(c->st);
    flags |= zgemm_algo_in_force() << 16;  // the captured sequence holds the kernels of this decomposition ...
    flags |= cgemm_variant_in_force() << 20;  // ... and of this complex64 GEMM kernel
    flags |= (pdl_enabled() ? 1 : 0) << 24;   // ... launched with or without programmatic dependent launch
    flags |= (lookahead_enabled() ? 1 : 0) << 25;  // ... with or without look-ahead forks
    hprmat_ctx::GraphEntry *ent = nullptr;
    for (auto &g : c->graphs)
        if (g.kind == kind && g.flags == flags && g.key == key) ent = &g;
    if (!ent) {
        hprmat_ctx::GraphEntry ne{kind, flags, key, nullptr, 0};
        const long long l0 = g_launches.load();
        if (cudaStreamBeginCapture(c->cap, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            const int rc = enqueue(c->cap);
            cudaGraph_t graph = nullptr;
            const cudaError_t e = cudaStreamEndCapture(c->cap, &graph);
            ne.launches = g_launches.load() - l0;
            g_launches.fetch_sub(ne.launches);  // captured, not launched
            if (rc == 0 && e == cudaSuccess && graph != nullptr) {
                if (cudaGraphInstantiate(&ne.exec, graph, 0) != cudaSuccess) ne.exec = nullptr;
            }
            if (graph) cudaGraphDestroy(graph);
        }
        cudaGetLastError();  // a refused capture is not an error of the solve
        c->graphs.push_back(ne);
        ent = &c->graphs.back();
    }
    if (!ent->exec) return enqueue(c->st);
    HP_CUDA(cudaGraphLaunch(ent->exec, c->st));
    g_launches.fetch_add(ent->launches);
    return 0;
}

template <class V> int getrs_replay(hprmat_ctx *c, int nrhs, V A, V B, LuWork<V> &wk, const void *key, int variant) {
    const int n = c->n;
    // the launch sequence depends on the right-hand-side count, the factored matrix and on whether the factorisation has
    // interchanges (speculate) or FP32-class products (accurate)
    const int flags = ((nrhs * 4 + variant) * 2 + (wk.speculate ? 1 : 0)) * 2 + (wk.accurate ? 1 : 0);
    return replay(c, 1, flags, key, [&](cudaStream_t s) { return getrs<V>(s, n, nrhs, A, B, wk); });
}

// ---- stages ---------------------------------------------------------------------------------------------------------------
int assemble(hprmat_ctx *c, Fac fac, const Problem &p, double energy, bool want_anorm) {
    cudaStream_t st = c->st;
    const int N = c->n, nch = c->nch, nb = c->nb;
    HP_CUDA(cudaMemsetAsync(c->d_info, 0, sizeof(int) * IN_NWORDS, st));
    if (p.W) HP_CUDA(cudaMemsetAsync(c->d_V, 0, sizeof(double2) * (size_t)nb * nch * nch, st));  // "no local potential"
    else HP_TRY(coupling_without_diagonal(st, c->tab, p.V, c->d_Voff));  // operand of the residual's tensor-core part
    if (fac == FAC_T3) {
        HP_TRY(type3_assemble(st, c->tab, c->d_KTinv, c->d_cf, energy, p.V, CView(c->d_Sre, c->d_Sim, c->ldS)));
    } else if (fac == FAC_C_Z) {
        if (p.W) HP_TRY(assemble_nonlocal(st, c->tab, energy, p.W, p.ldw, c->d_C, N));
        else HP_TRY(assemble_z(st, c->tab, energy, p.V, c->d_C, N));
    } else {
        HP_TRY(precond_invert(st, c->tab, energy, p.V, c->d_Kinv, c->d_info + IN_KBLOCK_SINGULAR, p.W, p.ldw));
        if (fac == FAC_S_Z) {
            if (p.W) {
                HP_TRY(zgemm_batched(st, nb, N, nb, 1.0, c->d_Kinv, nb, (long)nb * nb, p.W, p.ldw, nb, 0.0, c->d_C, N, nb, nch));
                const long tot = (long)nch * nb * nb;
                set_diag_blocks_identity_kernel<<<(int)std::min<long>((tot + 255) / 256, 148 * 8), 256, 0, st>>>(nch, nb, c->d_C, N);
                HP_LAUNCHED();
            } else {
                HP_TRY(precond_assemble_z(st, c->tab, c->d_Kinv, p.V, ZView(c->d_C, N)));
            }
        } else {
            CView S(c->d_Sre, c->d_Sim, c->ldS);
            if (p.W) HP_TRY(precond_assemble_nonlocal(st, c->tab, c->d_Kinv, p.W, p.ldw, S, c->d_Rlo, N));
            else HP_TRY(precond_assemble(st, c->tab, c->d_Kinv, p.V, S));
        }
    }
    if (want_anorm && p.W) HP_TRY(nonlocal_anorm(st, c->tab, energy, p.W, p.ldw, (double *)c->d_Rlo, c->d_scal + SC_ANORM));
    return 0;
}

int factor(hprmat_ctx *c, Fac fac, bool pivoting_fallback) {
    cudaStream_t st = c->st;
    const int N = c->n;
    int *zp = c->d_info + IN_ZERO_PIVOT;
    (void)st;
    if (fac == FAC_T3) {
        c->wc.speculate = false;
        c->wc.accurate = true;
        const int rc = replay(c, 0, 8, nullptr, [&](cudaStream_t s) {
            return getrf<CView>(s, N, CView(c->d_Sre, c->d_Sim, c->ldS), c->d_ipiv, zp, c->wc);
        });
        c->wc.accurate = false;
        return rc;
    }
    if (fac == FAC_S_C) {
        c->wc.speculate = !pivoting_fallback;
        return replay(c, 0, 4 + (pivoting_fallback ? 1 : 0), nullptr, [&](cudaStream_t s) {
            return getrf<CView>(s, N, CView(c->d_Sre, c->d_Sim, c->ldS), c->d_ipiv, zp, c->wc);
        });
    }
    c->wz.speculate = (fac == FAC_S_Z);
    return replay(c, 0, fac == FAC_S_Z ? 2 : 0, nullptr,
                  [&](cudaStream_t s) { return getrf<ZView>(s, N, ZView(c->d_C, N), c->d_ipiv, zp, c->wz); });
}

// X <- (factored matrix)^-1 (its right-hand sides); leaves max|X| in scal[SC_X0] (FP64) or scal[SC_XN] (complex64 factors)
int first_solve(hprmat_ctx *c, Fac fac, int *x0_word) {
    cudaStream_t st = c->st;
    const int N = c->n, nch = c->nch;
    if (fac == FAC_T3) {
        CView S(c->d_Sre, c->d_Sim, c->ldS), Bs(c->d_Bre, c->d_Bim, c->ldS);
        HP_TRY(type3_rhs(st, c->tab, c->d_g, Bs));
        c->wc.accurate = true;
        const int rc = getrs_replay<CView>(c, nch, S, Bs, c->wc, Bs.re, 2);
        c->wc.accurate = false;
        HP_TRY(rc);
        HP_TRY(type3_promote(st, c->tab, Bs, c->d_X, N, c->d_scal + SC_DN));
        *x0_word = SC_XN;
        return 0;
    }
    if (fac == FAC_S_C) {
        CView S(c->d_Sre, c->d_Sim, c->ldS), Bs(c->d_Bre, c->d_Bim, c->ldS);
        HP_TRY(precond_rhs(st, c->tab, c->d_Kinv, Bs));
        HP_TRY(getrs_replay<CView>(c, nch, S, Bs, c->wc, Bs.re, 0));
        HP_TRY(promote_add(st, N, nch, c->d_X, N, Bs, false, c->d_scal + SC_DN));
        *x0_word = SC_XN;
        return 0;
    }
    ZView A(c->d_C, N), X(c->d_X, N);
    if (fac == FAC_S_Z) HP_TRY(precond_rhs_z(st, c->tab, c->d_Kinv, X));
    else HP_TRY(build_rhs(st, c->tab, c->d_X, N));
    HP_TRY(getrs_replay<ZView>(c, nch, A, X, c->wz, X.p, fac));
    HP_TRY(maxabs(st, N, nch, c->d_X, N, c->d_scal + SC_X0));
    *x0_word = SC_X0;
    return 0;
}

// Rr <- B - (C - E I) X.  Local potentials: matrix-free, double-double accumulation (exact to the rounding of the result).
// Non-local: [structured part with V = 0, double-double] - W X on the FP64 tensor cores (working precision, reading R15).
int residual(hprmat_ctx *c, const Problem &p, double energy, double *rmax_dev) {
    cudaStream_t st = c->st;
    const int N = c->n, nch = c->nch;
    if (!p.W)
        return structured_residual_tc(st, c->tab, energy, p.V, c->d_Voff, c->d_X, N, c->d_Rr, c->d_Rlo, N, c->d_Xp, c->d_Pp,
                                      rmax_dev);
    HP_TRY(structured_residual_tc(st, c->tab, energy, c->d_V, nullptr, c->d_X, N, c->d_Rr, c->d_Rlo, N, nullptr, nullptr, nullptr));
    HP_TRY(gemm(st, N, nch, N, -1.0, ZView((double2 *)p.W, p.ldw), ZView(c->d_X, N), 1.0, ZView(c->d_Rr, N)));
    if (rmax_dev) HP_TRY(maxabs(st, N, nch, c->d_Rr, N, rmax_dev));
    return 0;
}

// X += (factored matrix)^-1 [K_d^-1] Rr, unless the device-side stopping rule has already fired
int correction(hprmat_ctx *c, Fac fac) {
    cudaStream_t st = c->st;
    const int N = c->n, nch = c->nch, nb = c->nb;
    const int *gate = c->d_info + IN_VERDICT;
    if (fac == FAC_C_Z) {
        HP_TRY(getrs_replay<ZView>(c, nch, ZView(c->d_C, N), ZView(c->d_Rr, N), c->wz, c->d_Rr, fac));
        return axpy_norm(st, N, nch, c->d_X, N, c->d_Rr, N, c->d_scal + SC_DN, gate);
    }
    // z = K_d^-1 r: one nb x nb by nb x nch product per channel (FP64 tensor cores), into Rlo
    HP_TRY(zgemm_batched(st, nb, nch, nb, 1.0, c->d_Kinv, nb, (long)nb * nb, c->d_Rr, N, nb, 0.0, c->d_Rlo, N, nb, nch));
    if (fac == FAC_S_Z) {
        HP_TRY(getrs_replay<ZView>(c, nch, ZView(c->d_C, N), ZView(c->d_Rlo, N), c->wz, c->d_Rlo, fac));
        return axpy_norm(st, N, nch, c->d_X, N, c->d_Rlo, N, c->d_scal + SC_DN, gate);
    }
    CView S(c->d_Sre, c->d_Sim, c->ldS), Bs(c->d_Bre, c->d_Bim, c->ldS);
    HP_TRY(demote(st, N, nch, c->d_Rlo, N, Bs));
    HP_TRY(getrs_replay<CView>(c, nch, S, Bs, c->wc, Bs.re, 0));
    return promote_add(st, N, nch, c->d_X, N, Bs, true, c->d_scal + SC_DN, gate);
}

int refine_step(hprmat_ctx *c, Fac fac, const Problem &p, double energy, double tol) {
    HP_TRY(residual(c, p, energy, nullptr));
    HP_TRY(correction(c, fac));
    refine_verdict_kernel<<<1, 1, 0, c->st>>>(c->d_scal, c->d_info, tol);
    HP_LAUNCHED();
    return 0;
}

// backward error of the returned X (definition in DESIGN.md reading R8), everything enqueued, nothing read back here
int report(hprmat_ctx *c, const Problem &p, double energy) {
    cudaStream_t st = c->st;
    HP_TRY(residual(c, p, energy, c->d_scal + SC_RMAX));
    if (!p.W) HP_TRY(structured_anorm(st, c->tab, energy, p.V, c->d_scal + SC_ANORM));
    return backward_error(st, c->n, c->nch, c->d_Rr, c->n, c->d_X, c->n, c->d_scal + SC_ANORM, c->d_scal + SC_BNORM,
                          c->d_scal + SC_BERR);
}

int read_back(hprmat_ctx *c) {
    HP_CUDA(cudaMemcpyAsync(c->h_scal, c->d_scal, sizeof(double) * SC_NWORDS, cudaMemcpyDeviceToHost, c->st));
    HP_CUDA(cudaMemcpyAsync(c->h_info, c->d_info, sizeof(int) * IN_NWORDS, cudaMemcpyDeviceToHost, c->st));
    HP_CUDA(cudaStreamSynchronize(c->st));
    return 0;
}

// status of a finished solve from the device words (host copies in h_scal / h_info); pivot_index out
int decode_status(const hprmat_ctx *c, Fac fac, bool must_converge, bool pivoting_fallback, int max_refine, bool have_berr,
                  int *pivot_index) {
    const int *hi = c->h_info;
    const double *hs = c->h_scal;
    *pivot_index = 0;
    const bool verified_fac = (fac == FAC_S_Z) || (fac == FAC_S_C && !pivoting_fallback);
    if (verified_fac && hi[IN_REFUTED] != 0) return UNUSABLE;
    if (hi[IN_ZERO_PIVOT] != 0 || ((fac == FAC_S_Z || fac == FAC_S_C) && hi[IN_KBLOCK_SINGULAR] != 0)) {
        if (fac == FAC_S_Z) return UNUSABLE;  // e.g. E on a pole of an uncoupled channel: C - E I itself may be regular
        *pivot_index = hi[IN_ZERO_PIVOT] ? hi[IN_ZERO_PIVOT] : hi[IN_KBLOCK_SINGULAR];
        return HPRMAT_ESINGULAR;
    }
    const double dn = hs[SC_DN_LAST], xn = hs[SC_XN_LAST];
    const int v = hi[IN_VERDICT];
    if (fac == FAC_S_Z) {
        // a correction that stopped shrinking while still large: the preconditioner is ill-conditioned at this energy
        if (max_refine > 0 && v != REF_CONTINUE && !(dn <= 1e-9 * xn)) return UNUSABLE;
        if (have_berr && !(hs[SC_BERR] <= 50.0 * c->n * 1.1102230246251565e-16)) return UNUSABLE;
    }
    if (must_converge && max_refine > 0) {
        if (v == REF_CONVERGED) return HPRMAT_OK;
        // a correction at the FP64 rounding floor of X is convergence, not failure
        if (v == REF_STAGNATED && dn <= 64.0 * 2.220446049250313e-16 * xn) return HPRMAT_OK;
        return HPRMAT_ENOTCONVERGED;  // stagnated above the floor, or max_refine steps were not enough
    }
    return HPRMAT_OK;  // FP64 modes: a stagnated correction is the rounding floor, not a failure
}

int run(hprmat_ctx *c, Fac fac, const Problem &p, double energy, int mode, int max_refine, double tol, double2 *R,
        hprmat_info *info, bool pivoting_fallback) {
    cudaStream_t st = c->st;
    const bool sync = info != nullptr;
    const bool mixed = fac == FAC_S_C || fac == FAC_T3;
    const bool must_converge = mode == HPRMAT_MIXED_REFINE;
    if (max_refine < 0) max_refine = mixed ? 5 : 2;
    if (mode == HPRMAT_MIXED || mode == HPRMAT_TYPE3) max_refine = 0;
    if (!(tol > 0.0)) tol = mixed ? 1e-12 : 1e-13;  // estimated relative error left in X; the north-star asks 1e-10 of R
    ScopedZgemmAlgo algo_scope(c->zgemm_algo);

    HP_CUDA(cudaEventRecord(c->ev[0], st));
    if (!c->reuse_factor) HP_TRY(assemble(c, fac, p, energy, sync));
    HP_CUDA(cudaEventRecord(c->ev[1], st));
    if (!c->reuse_factor) HP_TRY(factor(c, fac, pivoting_fallback));
    HP_CUDA(cudaEventRecord(c->ev[2], st));
    int x0_word = SC_X0;
    HP_TRY(first_solve(c, fac, &x0_word));
    HP_CUDA(cudaEventRecord(c->ev[3], st));
    int enq = 0;
    if (max_refine > 0) {
        refine_begin_kernel<<<1, 1, 0, st>>>(c->d_scal, c->d_info, x0_word);
        HP_LAUNCHED();
        // as many steps as the previous solve in this mode needed go out before anything is read back; a step enqueued
        // after the stopping rule has fired leaves X alone (gated update).  Unsynchronised calls get one spare step.
        int plan = std::max(1, c->plan_steps[mode]);
        if (!sync) plan = mixed ? plan + 1 : max_refine;
        plan = std::min(plan, max_refine);
        for (; enq < plan; ++enq) HP_TRY(refine_step(c, fac, p, energy, tol));
    }
    HP_CUDA(cudaEventRecord(c->ev[4], st));
    HP_TRY(contract(st, c->tab, c->d_X, c->n, R));
    HP_CUDA(cudaEventRecord(c->ev[5], st));
    c->have_x = true;
    c->last_fac = fac;
    c->last_fallback = pivoting_fallback;
    c->last_mode = mode;
    c->last_max_refine = max_refine;
    c->last_valid = true;
    if (!sync) return HPRMAT_OK;  // the status stays on the device: hprmat_last_status

    HP_TRY(report(c, p, energy));
    HP_TRY(read_back(c));
    bool extra = false;
    while (max_refine > 0 && c->h_info[IN_VERDICT] == REF_CONTINUE && enq < max_refine && c->h_info[IN_REFUTED] == 0 &&
           c->h_info[IN_ZERO_PIVOT] == 0 && c->h_info[IN_KBLOCK_SINGULAR] == 0) {
        // the prediction was short (first solve of a scan, or harder physics than the last point): one step at a time
        HP_TRY(refine_step(c, fac, p, energy, tol));
        ++enq;
        extra = true;
        HP_TRY(read_back(c));
    }
    if (extra) {
        HP_CUDA(cudaEventRecord(c->ev[4], st));
        HP_TRY(contract(st, c->tab, c->d_X, c->n, R));
        HP_CUDA(cudaEventRecord(c->ev[5], st));
        HP_TRY(report(c, p, energy));
        HP_TRY(read_back(c));
    }
    int pivot_index = 0;
    const int status = decode_status(c, fac, must_converge, pivoting_fallback, max_refine, true, &pivot_index);
    if (status == UNUSABLE) return UNUSABLE;
    if (max_refine > 0 && status == HPRMAT_OK) c->plan_steps[mode] = std::max(1, c->h_info[IN_STEPS]);
    info->status = status;
    info->refine_steps = c->h_info[IN_STEPS];
    info->pivot_index = pivot_index;
    info->reserved = c->h_info[IN_REFUTED];
    info->resid_max = c->h_scal[SC_RMAX];
    info->backward_err = status == HPRMAT_ESINGULAR ? -1.0 : c->h_scal[SC_BERR];
    info->ms_assemble = ev_ms(c->ev[0], c->ev[1]);
    info->ms_lu = ev_ms(c->ev[1], c->ev[2]);
    info->ms_solve = ev_ms(c->ev[2], c->ev[3]);
    info->ms_refine = ev_ms(c->ev[3], c->ev[4]);
    info->ms_contract = ev_ms(c->ev[4], c->ev[5]);
    info->ms_total = ev_ms(c->ev[0], c->ev[5]);
    info->lu_tflops = info->ms_lu > 0 ? (8.0 / 3.0) * (double)c->n * c->n * c->n / (info->ms_lu * 1e-3) * 1e-12 : 0.0;
    return status;
}

std::atomic<int> g_fp64_algo{2};  // process default of hprmat_fp64_algo; a context may carry its own (hprmat_set_option)

int solve_any(hprmat_ctx *c, const Problem &p, double energy, int mode, int max_refine, double tol, double2 *R, hprmat_info *info) {
    if (info) {
        *info = hprmat_info();
        info->backward_err = -1.0;
    }
    const int algo = c->fp64_algo ? c->fp64_algo : g_fp64_algo.load();
    Fac fac = mode == HPRMAT_FP64 ? (algo == 2 ? FAC_S_Z : FAC_C_Z) : mode == HPRMAT_TYPE3 ? FAC_T3 : FAC_S_C;
    int rc = run(c, fac, p, energy, mode, max_refine, tol, R, info, false);
    if (rc == UNUSABLE) {  // only reachable from a synchronised call: redo with pivoting
        *info = hprmat_info();
        info->backward_err = -1.0;
        const int refuted = c->h_info[IN_REFUTED];
        if (fac == FAC_S_Z) rc = run(c, FAC_C_Z, p, energy, mode, max_refine, tol, R, info, false);
        else rc = run(c, FAC_S_C, p, energy, mode, max_refine, tol, R, info, true);
        if (rc == UNUSABLE) rc = HPRMAT_ECUDA;  // cannot happen: neither fallback is a verified factorisation
        info->reserved = refuted;               // how many block panels refuted the diagonal (0: another reason)
    }
    if (info) info->status = rc;
    return rc;
}

}  // namespace

extern "C" int hprmat_solve_nonlocal(hprmat_ctx *ctx, double energy, const void *W, long ldw, int mode, int max_refine,
                                     double tol, void *R, hprmat_info *info) {
    if (!ctx) return -1;
    if (!W) return -3;
    if (ldw < ctx->n) return -4;
    if (mode != HPRMAT_FP64 && mode != HPRMAT_MIXED && mode != HPRMAT_MIXED_REFINE) return -5;
    if (!(ctx->max_mode & (1 << mode))) return -5;
    if (!R) return -8;
    Problem p;
    p.V = ctx->d_V;
    p.W = (const double2 *)W;
    p.ldw = ldw;
    return solve_any(ctx, p, energy, mode, max_refine, tol, (double2 *)R, info);
}

extern "C" int hprmat_fp64_algo(int algo) {
    if (algo == 1 || algo == 2) g_fp64_algo.store(algo);
    return g_fp64_algo.load();
}

extern "C" int hprmat_set_option(hprmat_ctx *ctx, int option, int value) {
    if (!ctx) return -1;
    switch (option) {
        case HPRMAT_OPT_FP64_ALGO:
            if (value != 0 && value != 1 && value != 2) return -3;
            ctx->fp64_algo = value;
            return HPRMAT_OK;
        case HPRMAT_OPT_ZGEMM_ALGO:
            if (value != 0 && value != 3 && value != 4) return -3;
            ctx->zgemm_algo = value;
            return HPRMAT_OK;
        case HPRMAT_OPT_GRAPHS:
            if (value != 0 && value != 1) return -3;
            ctx->use_graphs = value;
            return HPRMAT_OK;
        default: return -2;
    }
}

extern "C" int hprmat_solve(hprmat_ctx *ctx, double energy, const void *V, int mode, int max_refine, double tol, void *R,
                            hprmat_info *info) {
    if (!ctx) return -1;
    if (!V) return -3;
    if (mode != HPRMAT_FP64 && mode != HPRMAT_MIXED && mode != HPRMAT_MIXED_REFINE && mode != HPRMAT_TYPE3) return -4;
    if (!(ctx->max_mode & (1 << mode))) return -4;
    if (!R) return -7;
    Problem p;
    p.V = (const double2 *)V;
    return solve_any(ctx, p, energy, mode, max_refine, tol, (double2 *)R, info);
}

// measurement aid (include/hprmat_profile.h): how many launch sequences of this context are replayed from CUDA graphs and how
// many had to stay plain launches
extern "C" int hprmat_profile_graphs(const hprmat_ctx *ctx, int *captured, int *eager) {
    if (!ctx) return -1;
    int nc = 0, ne = 0;
    for (const auto &g : ctx->graphs) (g.exec ? nc : ne)++;
    if (captured) *captured = nc;
    if (eager) *eager = ne;
    return HPRMAT_OK;
}

// Sector matrices of a sub-interval context (propagate.cu; reading R16): one factorisation, two sets of nch
// right-hand sides (surface vectors of the right and of the left end), four contractions.
extern "C" int hprmat_solve_sector(hprmat_ctx *ctx, double energy, const void *V, int mode, int max_refine, double tol,
                                   void *Rsec, hprmat_info *info) {
    if (!ctx || !ctx->sector) return -1;
    if (!V) return -3;
    if (mode != HPRMAT_FP64 && mode != HPRMAT_MIXED && mode != HPRMAT_MIXED_REFINE) return -4;
    if (!(ctx->max_mode & (1 << mode))) return -4;
    if (!Rsec) return -7;
    if (!info) return -8;  // two dependent passes: the call is synchronised
    const long nn = (long)ctx->nch * ctx->nch;
    double2 *LL = (double2 *)Rsec, *LR = LL + nn, *RL = LL + 2 * nn, *RR = LL + 3 * nn;
    Problem p;
    p.V = (const double2 *)V;
    // pass 1: right-hand sides of the RIGHT end (tab.fa): X_R -> Rsec_RR, Rsec_LR
    int rc = solve_any(ctx, p, energy, mode, max_refine, tol, RR, info);
    if (rc != HPRMAT_OK && rc != HPRMAT_ENOTCONVERGED) return rc;
    HP_TRY(contract_with(ctx->st, ctx->tab, ctx->d_fa_left, ctx->d_X, ctx->n, LR));
    // pass 2: right-hand sides of the LEFT end, same factors: X_L -> Rsec_LL, Rsec_RL
    hprmat_info i2 = hprmat_info();
    double bn = 0.0;
    for (double f : ctx->fa_left) bn = std::max(bn, fabs(f));
    HP_CUDA(cudaMemcpyAsync(ctx->d_scal + SC_BNORM, &bn, sizeof(double), cudaMemcpyHostToDevice, ctx->st));
    const double *fa_right = ctx->tab.fa;
    ctx->tab.fa = ctx->d_fa_left;
    ctx->reuse_factor = true;
    int rc2 = run(ctx, (Fac)ctx->last_fac, p, energy, mode, max_refine, tol, LL, &i2, ctx->last_fallback);
    ctx->reuse_factor = false;
    ctx->tab.fa = fa_right;
    bn = 0.0;
    for (double f : ctx->fa) bn = std::max(bn, fabs(f));
    cudaMemcpyAsync(ctx->d_scal + SC_BNORM, &bn, sizeof(double), cudaMemcpyHostToDevice, ctx->st);
    if (rc2 == UNUSABLE) rc2 = HPRMAT_ENOTCONVERGED;  // the first pass accepted these factors; treat as not converged
    if (rc2 != HPRMAT_OK && rc2 != HPRMAT_ENOTCONVERGED) return rc2;
    HP_TRY(contract_with(ctx->st, ctx->tab, fa_right, ctx->d_X, ctx->n, RL));
    info->refine_steps = std::max(info->refine_steps, i2.refine_steps);
    info->resid_max = std::max(info->resid_max, i2.resid_max);
    info->backward_err = std::max(info->backward_err, i2.backward_err);
    info->ms_solve += i2.ms_solve;
    info->ms_refine += i2.ms_refine;
    info->ms_contract += i2.ms_contract;
    info->ms_total += i2.ms_total;
    rc = std::max(rc, rc2);
    info->status = rc;
    return rc;
}

// Status of the last solve of this context, for calls made with info == NULL: synchronises the stream, reads the device
// status words and decodes them exactly as a synchronised call would have.
extern "C" int hprmat_last_status(hprmat_ctx *ctx, int *refine_steps, int *pivot_index) {
    if (!ctx) return -1;
    if (!ctx->last_valid) return -1;
    HP_TRY(read_back(ctx));
    int piv = 0;
    int rc = decode_status(ctx, (Fac)ctx->last_fac, ctx->last_mode == HPRMAT_MIXED_REFINE, false, ctx->last_max_refine, false, &piv);
    if (rc == UNUSABLE) rc = HPRMAT_EUNVERIFIED;
    if (refine_steps) *refine_steps = ctx->h_info[IN_STEPS];
    if (pivot_index) *pivot_index = piv;
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
