// collision.cu -- hprmat_collision: collision matrix U of the open channels from the R-matrix at the channel radius
// ("matching to asymptotic solutions"), neutral and charged channels.
//
// The paper names the step and refers to its ref. [2]; the reading taken is DESIGN.md section 3, R14:
//     Z^O_cc' = (k_c' a)^-1/2 [ O_c delta_cc' - R_cc' (r dO_c'/dr)(a) ],     Z^I likewise with I_c,
//     U       = open rows of (Z^O)^-1 Z^I, columns restricted to the open channels,
// evaluated as U = 1 - 2i (Z^O)^-1 Z^F  (I = O - 2iF, so Z^I = Z^O - 2i Z^F): below a centrifugal barrier G/F reaches
// 1e30 and the literal form would lose F in the difference of two nearly equal columns,
// open channel (E > E_c):  O = G + iF, I = G - iF with the Coulomb wave functions F_l(eta_c, x), G_l(eta_c, x), x = k_c a,
// eta_c = Z1 Z2 e^2 / (2 h2m k_c) (eta = 0: the Riccati-Bessel functions x j_l(x), -x y_l(x));
// closed channel (E < E_c): no incoming wave, outgoing function replaced by the decaying Whittaker function
// W_{-eta_c, l+1/2}(2 kappa_c r) (eta = 0: x k_l(x), x = kappa_c a).
//
// Channel functions (host, long double).  eta = 0: Bessel recurrences.  eta != 0: Steed's method as described by Barnett
// (CF1 for F'/F at order l, downward recurrence to l = 0, CF2 for p + iq = (G' + iF')/(G + iF) at l = 0, Wronskian, upward
// recurrence of G); where q is small (under the Coulomb barrier, q < 1e-3 (|p| + |f|), where CF2 delivers it with few digits) F_0 comes from its
// power series (A&S 14.1.4-6, all terms of one sign there) and q from the Wronskian.  Closed channels: the continued
// fraction that CF2 becomes under k -> i kappa (real, derived in DESIGN.md section 3, R14).
//
// Host (long double): the 4 nch channel constants O, rO', I, rI' -- O(nch lmax) recurrences, the same kind of set-up
// work as the mesh tables of hprmat_setup.  Device: the two nch x nch matrices are built by one kernel from the device
// R, the linear system is solved by the library's own FP64 LU (getrf / getrs of lu.cu: DMMA GEMMs, cooperative panel), and
// a gather kernel extracts the open rows.  Nothing is synchronised; R never visits the host.
#include <cmath>
#include <vector>

#include "lu.cuh"

using namespace hp;

namespace {

typedef long double ld;

// Riccati-Bessel F_l(x) = x j_l(x) and x F_l'(x) for l = lmax only would do, but the recurrences deliver all l at once.
// j_l: Miller's downward recurrence from an order well above max(l, x), normalised on the larger of j_0, j_1 (stable for
// every x > 0); y_l and k_l: upward recurrences (stable: they are the dominant solutions).
struct ChannelFn {
    ld O_re, O_im, dO_re, dO_im;   // O and r dO/dr at r = a
    ld F, dF;                      // F and r dF/dr at r = a (open channels)
};

void bessel_j(int lmax, ld x, std::vector<ld> &j) {
    const int top = (int)std::max((ld)lmax, x) + 40 + (int)std::sqrt(40.0L * std::max((ld)lmax, x));
    std::vector<ld> t(top + 2, 0.0L);
    t[top + 1] = 0.0L;
    t[top] = 1e-280L;
    for (int l = top; l >= 1; --l) {
        t[l - 1] = (2.0L * l + 1.0L) / x * t[l] - t[l + 1];
        if (fabsl(t[l - 1]) > 1e250L)
            for (int m = l - 1; m <= top; ++m) t[m] *= 1e-250L;
    }
    const ld j0 = sinl(x) / x, j1 = sinl(x) / (x * x) - cosl(x) / x;
    const ld s = fabsl(j0) >= fabsl(j1) ? j0 / t[0] : j1 / t[1];
    j.resize(lmax + 2);
    for (int l = 0; l <= lmax + 1; ++l) j[l] = t[l] * s;
}

void bessel_y(int lmax, ld x, std::vector<ld> &y) {
    y.resize(lmax + 2);
    y[0] = -cosl(x) / x;
    y[1] = -cosl(x) / (x * x) - sinl(x) / x;
    for (int l = 1; l <= lmax; ++l) y[l + 1] = (2.0L * l + 1.0L) / x * y[l] - y[l - 1];
}

// modified spherical Bessel function of the second kind, k_l(x) = sqrt(pi / 2x) K_{l+1/2}(x), up to a factor common to all l
void bessel_k(int lmax, ld x, std::vector<ld> &k) {
    const ld h = 1.0L / x;  // the common factor (pi/2) exp(-x) is dropped: only the logarithmic derivative is used
    k.resize(lmax + 2);
    k[0] = h;
    k[1] = h * (1.0L + 1.0L / x);
    for (int l = 1; l <= lmax; ++l) k[l + 1] = k[l - 1] + (2.0L * l + 1.0L) / x * k[l];
}

// x d/dx [x f_l(x)] = x [ (l + 1) f_l(x) - x f_{l+1}(x) ] for f = j, y and k alike: f_l' = (l / x) f_l - f_{l+1} holds for
// all three (for k it follows from k_{l+1} = k_{l-1} + (2l + 1)/x k_l and k_l' = -k_{l-1} - (l + 1)/x k_l).
inline ld riccati_rderiv(int l, ld x, ld fl, ld fl1) { return x * ((l + 1.0L) * fl - x * fl1); }

const ld CF_EPS = 1e-19L, CF_TINY = 1e-300L;

inline ld cS(int k, ld eta, ld x) { return (ld)k / x + eta / (ld)k; }
inline ld cR2(int k, ld eta) { return 1.0L + (eta / (ld)k) * (eta / (ld)k); }

// F_l, G_l and x dF/dx, x dG/dx at (eta, x), eta != 0 or not.  false = a continued fraction or the series did not converge.
bool coulomb_fg(int l, ld eta, ld x, ld &F_out, ld &xdF_out, ld &G_out, ld &xdG_out) {
    // CF1 (modified Lentz): f = F_l'/F_l = S_{l+1} - R^2_{l+1} / (T_{l+1} - R^2_{l+2} / (T_{l+2} - ...)); sign of F_l from the
    // signs of the denominators
    ld f = cS(l + 1, eta, x);
    if (f == 0.0L) f = CF_TINY;
    ld C = f, D = 0.0L;
    int sign = 1;
    bool ok = false;
    for (long n = 1; n < 4000000; ++n) {
        const int k = l + (int)n;
        const ld a = -cR2(k, eta), b = (2.0L * k + 1.0L) * (1.0L / x + eta / ((ld)k * (k + 1.0L)));
        D = b + a * D;
        if (D == 0.0L) D = CF_TINY;
        C = b + a / C;
        if (C == 0.0L) C = CF_TINY;
        D = 1.0L / D;
        if (D < 0.0L) sign = -sign;
        const ld delta = C * D;
        f *= delta;
        if (fabsl(delta - 1.0L) < CF_EPS) { ok = true; break; }
    }
    if (!ok) return false;
    // downward recurrence of the unnormalised pair to l = 0
    const ld Fl = sign * 1e-30L, dFl = f * Fl;
    ld F = Fl, dF = dFl;
    for (int k = l; k >= 1; --k) {
        const ld Rk = sqrtl(cR2(k, eta)), Sk = cS(k, eta, x);
        const ld Fm = (Sk * F + dF) / Rk;
        dF = Sk * Fm - Rk * F;
        F = Fm;
        if (fabsl(F) > 1e2000L) return false;
    }
    ld f0 = dF / F;
    // CF2 at l = 0 (complex modified Lentz): p + iq = i (1 - eta/x) + (i/x) K,  K = ab / (2(x - eta + i) + (a+1)(b+1) / (2(x - eta + 2i) + ...)),
    // a = i eta, b = 1 + i eta
    ld hr = CF_TINY, hi = 0.0L, Cr = hr, Ci = 0.0L, Dr = 0.0L, Di = 0.0L;
    ok = false;
    for (long n = 1; n < 4000000; ++n) {
        // A = (a + n - 1)(b + n - 1) = (n - 1 + i eta)(n + i eta)
        const ld Ar = (ld)(n - 1) * (ld)n - eta * eta, Ai = eta * (2.0L * n - 1.0L);
        const ld Br = 2.0L * (x - eta), Bi = 2.0L * n;
        // D = 1 / (B + A D)
        ld tr = Br + Ar * Dr - Ai * Di, ti = Bi + Ar * Di + Ai * Dr;
        ld m = tr * tr + ti * ti;
        if (m == 0.0L) { tr = CF_TINY; m = tr * tr; }
        Dr = tr / m;
        Di = -ti / m;
        // C = B + A / C
        m = Cr * Cr + Ci * Ci;
        const ld qr = (Ar * Cr + Ai * Ci) / m, qi = (Ai * Cr - Ar * Ci) / m;
        Cr = Br + qr;
        Ci = Bi + qi;
        if (Cr == 0.0L && Ci == 0.0L) Cr = CF_TINY;
        const ld dr = Cr * Dr - Ci * Di, di = Cr * Di + Ci * Dr;
        const ld nr = hr * dr - hi * di, ni = hr * di + hi * dr;
        hr = nr;
        hi = ni;
        if (fabsl(dr - 1.0L) + fabsl(di) < CF_EPS) { ok = true; break; }
    }
    if (!ok) return false;
    const ld p = -hi / x;                       // i (1 - eta/x) + (i/x)(hr + i hi)
    ld q = (1.0L - eta / x) + hr / x;
    ld F0, G, dG;
    if (eta > 0.0L && q < 1e-3L * (fabsl(p) + fabsl(f0))) {
        // deep under the Coulomb barrier: F_0 = C_0(eta) sum_k A_k x^k, A_1 = 1, A_2 = eta, k(k-1) A_k = 2 eta A_{k-1} - A_{k-2}
        if (!(eta > 0.0L)) return false;
        const ld twopieta = 2.0L * acosl(-1.0L) * eta;
        const ld c0 = sqrtl(twopieta / expm1l(twopieta));
        ld Am2 = 1.0L, Am1 = eta, xp = x * x;
        ld s0 = x + eta * xp, s1 = 1.0L + 2.0L * eta * x;
        ok = false;
        for (int k = 3; k < 200000; ++k) {
            const ld Ak = (2.0L * eta * Am1 - Am2) / ((ld)k * (k - 1.0L));
            const ld xp1 = xp;
            xp *= x;
            const ld t0 = Ak * xp, t1 = (ld)k * Ak * xp1;
            s0 += t0;
            s1 += t1;
            Am2 = Am1;
            Am1 = Ak;
            if (fabsl(t0) < CF_EPS * fabsl(s0) && fabsl(t1) < CF_EPS * fabsl(s1)) { ok = true; break; }
        }
        if (!ok) return false;
        F0 = c0 * s0;
        f0 = s1 / s0;
        const ld d = f0 - p, u = F0 * F0;
        q = 2.0L * u * d * d / (1.0L + sqrtl(1.0L - 4.0L * u * u * d * d));   // the small root of u q^2 - q + u d^2 = 0
        G = d * F0 / q;
        dG = p * G - q * F0;
    } else {
        const ld gam = (f0 - p) / q;
        F0 = copysignl(1.0L / sqrtl((f0 - p) * gam + q), F);
        G = gam * F0;
        dG = (p * gam - q) * F0;
    }
    const ld scale = F0 / F;
    for (int k = 0; k < l; ++k) {
        const ld Rk = sqrtl(cR2(k + 1, eta)), Sk = cS(k + 1, eta, x);
        const ld Gp = (Sk * G - dG) / Rk;
        dG = Rk * G - Sk * Gp;
        G = Gp;
    }
    F_out = Fl * scale;
    xdF_out = x * dFl * scale;
    G_out = G;
    xdG_out = x * dG;
    return std::isfinite((double)F_out) && std::isfinite((double)G_out) && std::isfinite((double)xdG_out);
}

// r W'/W of the decaying Whittaker function W_{-eta, l+1/2}(2x):  -(x + eta) + ab / (2(x + eta + 1) - (a+1)(b+1) / (2(x + eta + 2) - ...)),
// a = eta - l, b = eta + l + 1 (terminates when eta - l is a non-positive integer, e.g. always for eta = 0)
bool whittaker_logderiv(int l, ld eta, ld x, ld &out) {
    const ld a = eta - (ld)l, b = eta + (ld)l + 1.0L;
    ld h = CF_TINY, C = h, D = 0.0L;
    if (a * b == 0.0L) { out = -(x + eta); return true; }
    for (long n = 1; n < 4000000; ++n) {
        const ld A = (n == 1) ? a * b : -(a + (ld)(n - 1)) * (b + (ld)(n - 1));
        const ld B = 2.0L * (x + eta + (ld)n);
        if (A == 0.0L) { out = -(x + eta) + h; return true; }
        D = B + A * D;
        if (D == 0.0L) D = CF_TINY;
        C = B + A / C;
        if (C == 0.0L) C = CF_TINY;
        D = 1.0L / D;
        const ld delta = C * D;
        h *= delta;
        if (fabsl(delta - 1.0L) < CF_EPS) { out = -(x + eta) + h; return true; }
    }
    return false;
}

bool channel_fn(int l, ld eta, ld x, bool open, ChannelFn &c) {
    c = ChannelFn();
    if (eta != 0.0L) {
        if (open) {
            ld F, dF, G, dG;
            if (!coulomb_fg(l, eta, x, F, dF, G, dG)) return false;
            c.O_re = G; c.O_im = F; c.dO_re = dG; c.dO_im = dF;
            c.F = F; c.dF = dF;
        } else {
            c.O_re = 1.0L;
            if (!whittaker_logderiv(l, eta, x, c.dO_re)) return false;
        }
        return true;
    }
    if (open) {
        std::vector<ld> j, y;
        bessel_j(l, x, j);
        bessel_y(l, x, y);
        const ld F = x * j[l], G = -x * y[l];
        const ld dF = riccati_rderiv(l, x, j[l], j[l + 1]), dG = -riccati_rderiv(l, x, y[l], y[l + 1]);
        c.O_re = G; c.O_im = F; c.dO_re = dG; c.dO_im = dF;
        c.F = F; c.dF = dF;
    } else {
        std::vector<ld> k;
        bessel_k(l, x, k);
        // scaling a column of Z^O rescales only the matching (closed) row of the solution, which is discarded: the column is
        // normalised to W = 1 so that deeply closed channels (W ~ exp(-kappa a)) cannot underflow
        c.O_re = 1.0L;
        c.dO_re = riccati_rderiv(l, x, k[l], k[l + 1]) / (x * k[l]);
    }
    return true;
}

// tab: [0, nch) O, [nch, 2nch) r dO/dr, [2nch, 3nch) F, [3nch, 4nch) r dF/dr, each already divided by sqrt(k_c a)
// ZO nch x nch (ld nch), ZI = Z^F nch x nopen (ld nch): column q of ZI belongs to channel open_idx[q]
__global__ void collision_matrices_kernel(int nch, int nopen, const double2 *__restrict__ R, const double2 *__restrict__ tab,
                                          const int *__restrict__ open_idx, double2 *__restrict__ ZO,
                                          double2 *__restrict__ ZI) {
    const long total = (long)nch * (nch + nopen);
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x) {
        const int row = (int)(idx % nch);
        const int colx = (int)(idx / nch);
        const bool incoming = colx >= nch;
        const int col = incoming ? open_idx[colx - nch] : colx;
        const double2 f = tab[(incoming ? 2 * nch : 0) + col], df = tab[(incoming ? 3 * nch : nch) + col];
        const double2 rv = R[(long)col * nch + row];
        double2 z = make_double2(-(rv.x * df.x - rv.y * df.y), -(rv.x * df.y + rv.y * df.x));
        if (row == col) {
            z.x += f.x;
            z.y += f.y;
        }
        if (incoming) ZI[(long)(colx - nch) * nch + row] = z;
        else ZO[(long)col * nch + row] = z;
    }
}

__global__ void gather_open_rows_kernel(int nch, int nopen, const double2 *__restrict__ X, const int *__restrict__ open_idx,
                                        double2 *__restrict__ U) {
    const long total = (long)nopen * nopen;
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x) {
        const int p = (int)(idx % nopen), q = (int)(idx / nopen);
        const double2 y = X[(long)q * nch + open_idx[p]];     // U = 1 - 2i Y on the open rows
        U[idx] = make_double2((p == q ? 1.0 : 0.0) + 2.0 * y.y, -2.0 * y.x);
    }
}

inline size_t up256(size_t b) { return (b + 255) & ~(size_t)255; }

}  // namespace

extern "C" size_t hprmat_collision_workspace_bytes(int nch) {
    if (nch < 0) return 0;
    const size_t n = (size_t)nch;
    return up256(4 * n * sizeof(double2)) + up256(n * sizeof(int)) + 2 * up256(n * n * sizeof(double2)) +
           up256(n * sizeof(int)) + 256 + LuWork<ZView>::bytes(nch);
}

extern "C" int hprmat_channel_functions(int l, double eta, double x, int open, double *out) {
    if (l < 0) return -1;
    if (!std::isfinite(eta)) return -2;
    if (!(x > 0.0) || !std::isfinite(x)) return -3;
    if (!out) return -5;
    ChannelFn c;
    if (!channel_fn(l, (ld)eta, (ld)x, open != 0, c)) return -3;
    out[0] = (double)c.F;
    out[1] = (double)c.dF;
    out[2] = (double)c.O_re;
    out[3] = (double)c.dO_re;
    return HPRMAT_OK;
}

extern "C" int hprmat_collision(void *cuda_stream, int nch, const int *lval, const double *ethr, const double *zze2,
                                double energy, double h2m, double a, const void *R, void *U, int *nopen_out, int *info_dev,
                                void *workspace, size_t workspace_bytes) {
    if (nch < 1) return -2;
    if (!lval) return -3;
    if (!ethr) return -4;
    if (!std::isfinite(energy)) return -6;
    if (!(h2m > 0.0)) return -7;
    if (!(a > 0.0)) return -8;
    if (!R) return -9;
    if (!nopen_out) return -11;
    if (!info_dev) return -12;
    if (!workspace || ((uintptr_t)workspace & 255)) return -13;
    if (workspace_bytes < hprmat_collision_workspace_bytes(nch)) return HPRMAT_ENOMEM;
    for (int c = 0; c < nch; ++c) {
        if (lval[c] < 0) return -3;
        if (energy == ethr[c]) return -6;  // exactly at a threshold: k_c = 0, the matching is undefined
        if (zze2 && !std::isfinite(zze2[c])) return -5;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;

    std::vector<double2> tab(4 * (size_t)nch);
    std::vector<int> open_idx;
    for (int c = 0; c < nch; ++c) {
        const bool open = energy > ethr[c];
        const ld x = sqrtl(fabsl((ld)energy - (ld)ethr[c]) / (ld)h2m) * (ld)a;
        const ld kc = x / (ld)a;
        const ld eta = zze2 ? (ld)zze2[c] / (2.0L * (ld)h2m * kc) : 0.0L;
        ChannelFn f;
        if (!channel_fn(lval[c], eta, x, open, f)) return -6;  // too close to a threshold for the continued fractions
        const ld s = 1.0L / sqrtl(x);
        tab[c] = make_double2((double)(f.O_re * s), (double)(f.O_im * s));
        tab[nch + c] = make_double2((double)(f.dO_re * s), (double)(f.dO_im * s));
        tab[2 * nch + c] = make_double2((double)(f.F * s), 0.0);
        tab[3 * nch + c] = make_double2((double)(f.dF * s), 0.0);
        if (open) open_idx.push_back(c);
    }
    const int nopen = (int)open_idx.size();
    *nopen_out = nopen;
    HP_CUDA(cudaMemsetAsync(info_dev, 0, sizeof(int), st));
    if (nopen == 0) return HPRMAT_OK;
    if (!U) return -10;

    char *p = (char *)workspace;
    double2 *d_tab = (double2 *)p;  p += up256(4 * (size_t)nch * sizeof(double2));
    int *d_open = (int *)p;         p += up256((size_t)nch * sizeof(int));
    double2 *d_ZO = (double2 *)p;   p += up256((size_t)nch * nch * sizeof(double2));
    double2 *d_ZI = (double2 *)p;   p += up256((size_t)nch * nch * sizeof(double2));
    int *d_ipiv = (int *)p;         p += up256((size_t)nch * sizeof(int)) + 256;
    LuWork<ZView> wk;
    wk.carve(p, nch);

    // pageable sources: cudaMemcpyAsync stages them before it returns, so the vectors may die at the end of this call
    HP_CUDA(cudaMemcpyAsync(d_tab, tab.data(), tab.size() * sizeof(double2), cudaMemcpyHostToDevice, st));
    HP_CUDA(cudaMemcpyAsync(d_open, open_idx.data(), (size_t)nopen * sizeof(int), cudaMemcpyHostToDevice, st));
    {
        ProfCat pc(PROF_OTHER);
        const long total = (long)nch * (nch + nopen);
        const int blocks = (int)std::min<long>((total + 255) / 256, 148 * 8);
        collision_matrices_kernel<<<blocks, 256, 0, st>>>(nch, nopen, (const double2 *)R, d_tab, d_open, d_ZO, d_ZI);
        HP_LAUNCHED();
    }
    HP_TRY(getrf<ZView>(st, nch, ZView(d_ZO, nch), d_ipiv, info_dev, wk));
    HP_TRY(getrs<ZView>(st, nch, nopen, ZView(d_ZO, nch), ZView(d_ZI, nch), wk));
    {
        ProfCat pc(PROF_OTHER);
        const long total = (long)nopen * nopen;
        const int blocks = (int)std::min<long>((total + 255) / 256, 148 * 8);
        gather_open_rows_kernel<<<blocks, 256, 0, st>>>(nch, nopen, d_ZI, d_open, (double2 *)U);
        HP_LAUNCHED();
    }
    return HPRMAT_OK;
}
