/*
 * hprmat_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU implementation of the hot path of the R-matrix method of
 * arxiv 2512.11590 (HPRMAT): assemble C - E*I (Eqs. 1-4), solve (C - E*I) X = B by LU with
 * partial pivoting and substitution (Eq. 5), R = (h2m/a) B^T X (PAPER.md:137 step 4, prefactor
 * from BASELINE.json north_star).  complex double storage, long double (x87, 64-bit mantissa) accumulation.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this.  It shares
 * no code with paper_2512_11590_b200/csrc (the CUDA path) and neither includes the other.
 *
 * Pins (tests/test_oracle_*.py, all "-m not gpu"): mesh -> quadrature exactness and numpy.polynomial leggauss;
 * fa, T -> explicit Lagrange polynomials integrated exactly in mpmath (T_ij = int f_i' f_j'); LU/solve -> Cramer's
 * rule and Gauss-Jordan inversion in mpmath for N <= 8, manufactured solution x = 1; whole chain ->
 * V = 0 and constant-well closed forms, R = R^T, S-matrix unitarity for real potentials.  No function here is
 * "parity unpinned".
 *
 * Readings of the paper where it is silent (DESIGN.md section 3 lists all of them):
 *  - mesh / f_i(a) / T_ij closed forms are the standard Lagrange-Legendre mesh regularised by r (the paper's refs
 *    [2],[3]; PAPER.md:79 only names them);
 *  - thresholds enter as +E_c on the diagonal (PAPER.md:75-77 hides them in "internal quantum numbers");
 *  - pivot = first row of maximal |re|+|im| (PAPER.md:127 says only "partial pivoting").
 *
 * Index convention (step 4): row/col of channel c (0-based), mesh point i (0-based) is c*nb + i.
 * All matrices column-major.  V[(i*nch + c2)*nch + c1] = V_{c1 c2}(r_i).
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double _Complex zc;
typedef long double ld;

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------------------------
 * Step 1 ("Gauss-Legendre quadrature points {r_i} with weights {lambda_i} on (0,a)").
 * t_i = roots of P_nb on (-1,1) by Newton in long double; x_i = (1+t_i)/2 ascending; r_i = a x_i;
 * lam_i = weights on (0,1) = 1/((1-t^2) P'(t)^2)  (the paper's lambda_i on (0,a) is a*lam_i);
 * fa_i = f_i(a) = (-1)^(nb+i) / sqrt(a x_i (1-x_i)), i = 1..nb  -- the paper's q2(r_i).
 * ---------------------------------------------------------------------------------------------------------- */
static void legendre_ld(int n, ld t, ld *pn, ld *pnm1) {
    ld p0 = 1.0L, p1 = t;
    if (n == 0) { *pn = 1.0L; *pnm1 = 0.0L; return; }
    for (int k = 2; k <= n; ++k) {
        ld p2 = ((2 * k - 1) * t * p1 - (k - 1) * p0) / k;
        p0 = p1; p1 = p2;
    }
    *pn = p1; *pnm1 = p0;
}

int orc_mesh(int nb, double a, double *x, double *lam, double *r, double *fa) {
    if (nb < 1 || !(a > 0)) return -1;
    const ld pi = 3.14159265358979323846264338327950288L;
    for (int i = 1; i <= nb; ++i) {
        /* i-th root counted from the right end t ~ +1 downwards; Chebyshev-like first guess */
        ld t = cosl(pi * (i - 0.25L) / (nb + 0.5L));
        ld pn, pnm1, dp = 0;
        for (int it = 0; it < 100; ++it) {
            legendre_ld(nb, t, &pn, &pnm1);
            dp = nb * (pnm1 - t * pn) / (1.0L - t * t);
            ld dt = pn / dp;
            t -= dt;
            if (fabsl(dt) < 1e-19L) break;
        }
        legendre_ld(nb, t, &pn, &pnm1);
        dp = nb * (pnm1 - t * pn) / (1.0L - t * t);
        int idx = nb - i; /* ascending order */
        ld xi = (1.0L + t) / 2.0L;
        ld li = 1.0L / ((1.0L - t * t) * dp * dp);
        x[idx] = (double)xi;
        lam[idx] = (double)li;
        r[idx] = (double)((ld)a * xi);
        int sgn = ((nb + (idx + 1)) % 2 == 0) ? 1 : -1;
        fa[idx] = (double)(sgn / sqrtl((ld)a * xi * (1.0L - xi)));
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * Step 2 ("K_alpha ... full n_lag x n_lag matrix including the Bloch operator boundary term").
 * T_ij = <f_i| -d^2/dr^2 + delta(r-a) d/dr |f_j> in units hbar^2/2mu = 1, on (0,a):
 *   T_ii = [(4n^2+4n+3) x_i(1-x_i) - 6x_i + 1] / [3 a^2 x_i^2 (1-x_i)^2]
 *   T_ij = (-1)^(i+j) / [a^2 sqrt(x_i x_j (1-x_i)(1-x_j))]
 *          * [n^2 + n + 1 + (x_i + x_j - 2 x_i x_j)/(x_i-x_j)^2 - 1/(1-x_i) - 1/(1-x_j)]
 * evaluated in long double from the double-rounded x_i, rounded once.  T column-major nb x nb (symmetric).
 * ---------------------------------------------------------------------------------------------------------- */
int orc_kinetic(int nb, double a, const double *x, double *T) {
    if (nb < 1 || !(a > 0)) return -1;
    ld n = nb, a2 = (ld)a * (ld)a;
    for (int j = 0; j < nb; ++j)
        for (int i = 0; i < nb; ++i) {
            ld xi = x[i], xj = x[j];
            ld v;
            if (i == j) {
                v = ((4 * n * n + 4 * n + 3) * xi * (1 - xi) - 6 * xi + 1) / (3 * a2 * xi * xi * (1 - xi) * (1 - xi));
            } else {
                ld s = ((i + j) % 2 == 0) ? 1.0L : -1.0L;
                ld d = xi - xj;
                v = s / (a2 * sqrtl(xi * xj * (1 - xi) * (1 - xj))) *
                    (n * n + n + 1 + (xi + xj - 2 * xi * xj) / (d * d) - 1 / (1 - xi) - 1 / (1 - xj));
            }
            T[(size_t)j * nb + i] = (double)v;
        }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * Step 3 (Eqs. 3-4; Eq. 1 for the diagonal terms).  C - E*I, N x N column-major:
 *   row = c*nb + i, col = c'*nb + j:
 *   delta_cc' [ h2m*T_ij + delta_ij ( h2m*l_c(l_c+1)/r_i^2 + E_c - E ) ] + delta_ij V_cc'(r_i)
 * FP64 evaluation order of the diagonal entry (reading R4):
 *   ((h2m*T_ii + h2m*l(l+1)/(r_i*r_i)) + (E_c - E)) + V_cc(r_i)
 * ---------------------------------------------------------------------------------------------------------- */
int orc_assemble(int nch, int nb, double a, double h2m, const int *lval, const double *ethr, double energy,
                 const zc *V, zc *C) {
    if (nch < 1 || nb < 1) return -1;
    size_t N = (size_t)nch * nb;
    double *x = malloc(sizeof(double) * nb * 4), *lam = x + nb, *r = x + 2 * nb, *fa = x + 3 * nb;
    double *T = malloc(sizeof(double) * nb * nb);
    if (!x || !T) return -2;
    orc_mesh(nb, a, x, lam, r, fa);
    orc_kinetic(nb, a, x, T);
    memset(C, 0, sizeof(zc) * N * N);
    for (int c2 = 0; c2 < nch; ++c2)
        for (int j = 0; j < nb; ++j) {
            size_t col = (size_t)c2 * nb + j;
            for (int c1 = 0; c1 < nch; ++c1) {
                if (c1 == c2) {
                    for (int i = 0; i < nb; ++i) {
                        size_t row = (size_t)c1 * nb + i;
                        volatile double kt = h2m * T[(size_t)j * nb + i];
                        if (i == j) {
                            double l = lval[c1];
                            volatile double cf = h2m * l * (l + 1) / (r[i] * r[i]);
                            volatile double d = kt + cf;
                            volatile double de = ethr[c1] - energy;
                            volatile double d2 = d + de;
                            C[col * N + row] = d2 + V[((size_t)i * nch + c2) * nch + c1];
                        } else {
                            C[col * N + row] = kt;
                        }
                    }
                } else {
                    size_t row = (size_t)c1 * nb + j;
                    C[col * N + row] = V[((size_t)j * nch + c2) * nch + c1];
                }
            }
        }
    free(x); free(T);
    return 0;
}

/* Step 4: B[(c,i), c'] = fa_i delta_cc'.  N x nch column-major. */
int orc_rhs(int nch, int nb, const double *fa, zc *B) {
    size_t N = (size_t)nch * nb;
    memset(B, 0, sizeof(zc) * N * nch);
    for (int c = 0; c < nch; ++c)
        for (int i = 0; i < nb; ++i) B[(size_t)c * N + (size_t)c * nb + i] = fa[i];
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * Accumulated complex dot product sum_k p[k]*q[k], both contiguous.  mode 0: long double; mode 1: double
 * ("big-N mode").  Returns through *sr,*si as long double.
 * ---------------------------------------------------------------------------------------------------------- */
static inline void cdot(const zc *p, const zc *q, size_t n, int mode, ld *sr, ld *si) {
    if (mode == 0) {
        ld ar = 0, ai = 0;
        for (size_t k = 0; k < n; ++k) {
            ld pr = creal(p[k]), pi = cimag(p[k]), qr = creal(q[k]), qi = cimag(q[k]);
            ar += pr * qr - pi * qi;
            ai += pr * qi + pi * qr;
        }
        *sr = ar; *si = ai;
    } else {
        double ar = 0, ai = 0;
        const double *pd = (const double *)p, *qd = (const double *)q;
        for (size_t k = 0; k < n; ++k) {
            double pr = pd[2 * k], pi = pd[2 * k + 1], qr = qd[2 * k], qi = qd[2 * k + 1];
            ar += pr * qr - pi * qi;
            ai += pr * qi + pi * qr;
        }
        *sr = ar; *si = ai;
    }
}

static inline zc cdiv_ld(ld ar, ld ai, zc p) {
    ld pr = creal(p), pi = cimag(p);
    ld den = pr * pr + pi * pi;
    return (double)((ar * pr + ai * pi) / den) + (double)((ai * pr - ar * pi) / den) * I;
}

/* ------------------------------------------------------------------------------------------------------------
 * Step 5 (Eq. 5): M = P L U, unit-diagonal L, partial pivoting.  Crout ordering so every
 * entry of L and U is  a_ij - sum_k l_ik u_kj  accumulated (long double in mode 0) and rounded ONCE:
 *   for j: (a) w_i = a_ij - sum_{k<j} l_ik u_kj, i >= j            (independent per row: the OpenMP loop)
 *          (b) p = first argmax_i |re w_i| + |im w_i|; swap rows j,p (whole rows); ipiv[j] = p
 *          (c) u_jc = a_jc - sum_{k<j} l_jk u_kc, c > j              (independent per column)
 *          (d) l_ij = w_i / u_jj, i > j
 * Storage: W row-major n x n (holds A, then L below / U on and above the diagonal); Uc[c*n + k] = u_kc is a
 * column-contiguous copy of U so both dot products run over contiguous memory.
 * Returns 0, or j+1 if the j-th pivot is exactly zero.
 * ---------------------------------------------------------------------------------------------------------- */
typedef struct { size_t n; zc *W; zc *Uc; int *ipiv; } orc_lu;

static int lu_factor(orc_lu *f, int mode) {
    size_t n = f->n;
    zc *W = f->W, *Uc = f->Uc;
    int info = 0;
    for (size_t j = 0; j < n; ++j) {
        /* (a) */
#pragma omp parallel for schedule(static) if (n - j > 64)
        for (size_t i = j; i < n; ++i) {
            ld sr, si;
            cdot(W + i * n, Uc + j * n, j, mode, &sr, &si);
            zc aij = W[i * n + j];
            W[i * n + j] = (double)((ld)creal(aij) - sr) + (double)((ld)cimag(aij) - si) * I;
        }
        /* (b) */
        size_t p = j; double best = -1.0;
        for (size_t i = j; i < n; ++i) {
            double m = fabs(creal(W[i * n + j])) + fabs(cimag(W[i * n + j]));
            if (m > best) { best = m; p = i; }
        }
        f->ipiv[j] = (int)p;
        if (p != j)
            for (size_t k = 0; k < n; ++k) { zc t = W[j * n + k]; W[j * n + k] = W[p * n + k]; W[p * n + k] = t; }
        zc piv = W[j * n + j];
        Uc[j * n + j] = piv;
        if (best == 0.0) { if (!info) info = (int)j + 1; continue; }
        /* (c) */
#pragma omp parallel for schedule(static) if (n - j > 64)
        for (size_t c = j + 1; c < n; ++c) {
            ld sr, si;
            cdot(W + j * n, Uc + c * n, j, mode, &sr, &si);
            zc a = W[j * n + c];
            zc u = (double)((ld)creal(a) - sr) + (double)((ld)cimag(a) - si) * I;
            W[j * n + c] = u;
            Uc[c * n + j] = u;
        }
        /* (d) */
        for (size_t i = j + 1; i < n; ++i) W[i * n + j] = cdiv_ld(creal(W[i * n + j]), cimag(W[i * n + j]), piv);
    }
    return info;
}

/* Step 6 ("forward and backward substitution"): X <- U^-1 L^-1 P X, nrhs columns, column-major ldx=n.
 * Each x_i is one accumulated dot product (row of L / row of U, contiguous in W) rounded once. */
static void lu_solve(const orc_lu *f, zc *X, size_t nrhs, int mode) {
    size_t n = f->n;
    const zc *W = f->W;
#pragma omp parallel for schedule(dynamic, 1)
    for (size_t c = 0; c < nrhs; ++c) {
        zc *x = X + c * n;
        for (size_t j = 0; j < n; ++j) {
            size_t p = (size_t)f->ipiv[j];
            if (p != j) { zc t = x[j]; x[j] = x[p]; x[p] = t; }
        }
        for (size_t i = 0; i < n; ++i) {
            ld sr, si;
            cdot(W + i * n, x, i, mode, &sr, &si);
            x[i] = (double)((ld)creal(x[i]) - sr) + (double)((ld)cimag(x[i]) - si) * I;
        }
        for (size_t ii = n; ii-- > 0;) {
            ld sr, si;
            cdot(W + ii * n + ii + 1, x + ii + 1, n - ii - 1, mode, &sr, &si);
            x[ii] = cdiv_ld((ld)creal(x[ii]) - sr, (ld)cimag(x[ii]) - si, W[ii * n + ii]);
        }
    }
}

static int lu_alloc(orc_lu *f, size_t n) {
    f->n = n;
    f->W = malloc(sizeof(zc) * n * n);
    f->Uc = malloc(sizeof(zc) * n * n);
    f->ipiv = malloc(sizeof(int) * n);
    return (f->W && f->Uc && f->ipiv) ? 0 : -2;
}
static void lu_free(orc_lu *f) { free(f->W); free(f->Uc); free(f->ipiv); }

/* ------------------------------------------------------------------------------------------------------------
 * Dense solve A X = B (the paper's ZGESV call, PAPER.md:127,137 step 3).  A n x n, B and X n x nrhs, column-major,
 * A and B are not modified.  nrefine steps of iterative refinement with the residual B - A X accumulated in long
 * double from the ORIGINAL A (PAPER.md:151 describes the scheme; here it only sharpens the oracle itself).
 * ipiv_out (may be NULL): 0-based pivot rows.  Returns 0, >0 singular pivot index, <0 bad argument / no memory.
 * ---------------------------------------------------------------------------------------------------------- */
int orc_solve(int n_, int nrhs_, const zc *A, const zc *B, zc *X, int *ipiv_out, int mode, int nrefine) {
    if (n_ < 0 || nrhs_ < 0) return -1;
    size_t n = n_, nrhs = nrhs_;
    if (n == 0 || nrhs == 0) return 0;
    orc_lu f;
    if (lu_alloc(&f, n)) return -2;
    for (size_t i = 0; i < n; ++i)
        for (size_t j = 0; j < n; ++j) f.W[i * n + j] = A[j * n + i];
    int info = lu_factor(&f, mode);
    if (ipiv_out) memcpy(ipiv_out, f.ipiv, sizeof(int) * n);
    if (info) { lu_free(&f); return info; }
    memcpy(X, B, sizeof(zc) * n * nrhs);
    lu_solve(&f, X, nrhs, mode);
    zc *Rr = malloc(sizeof(zc) * n * nrhs);
    /* row-major copy of A for contiguous residual rows */
    for (size_t i = 0; i < n; ++i)
        for (size_t j = 0; j < n; ++j) f.Uc[i * n + j] = A[j * n + i];
    for (int it = 0; it < nrefine; ++it) {
#pragma omp parallel for schedule(static) collapse(2)
        for (size_t c = 0; c < nrhs; ++c)
            for (size_t i = 0; i < n; ++i) {
                ld sr, si;
                cdot(f.Uc + i * n, X + c * n, n, 0, &sr, &si);
                Rr[c * n + i] = (double)((ld)creal(B[c * n + i]) - sr) + (double)((ld)cimag(B[c * n + i]) - si) * I;
            }
        lu_solve(&f, Rr, nrhs, mode);
        for (size_t k = 0; k < n * nrhs; ++k) X[k] += Rr[k];
    }
    free(Rr);
    lu_free(&f);
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * Structured (matrix-free) residual  Rr = B - (C - E I) X  in long double, from the block structure of Eqs. 3-4:
 *   r[(c,i), q] = fa_i delta_cq - sum_j h2m T_ij X[(c,j),q] - (h2m l_c(l_c+1)/r_i^2 + E_c - E) X[(c,i),q]
 *                 - sum_c' V_cc'(r_i) X[(c',i),q]
 * X, Rr: N x nrhs column-major; B is implied (nrhs must be nch) when Bx == NULL, else Bx is used.
 * Also used by tests as the a-posteriori certificate on a solution computed elsewhere (it only evaluates a residual).
 * ---------------------------------------------------------------------------------------------------------- */
int orc_structured_residual(int nch, int nb, double a, double h2m, const int *lval, const double *ethr, double energy,
                            const zc *V, int nrhs, const zc *Bx, const zc *X, zc *Rr) {
    size_t N = (size_t)nch * nb;
    double *x = malloc(sizeof(double) * nb * 4), *lam = x + nb, *r = x + 2 * nb, *fa = x + 3 * nb;
    double *T = malloc(sizeof(double) * nb * nb);
    if (!x || !T) return -2;
    if (!Bx && nrhs != nch) return -1;
    orc_mesh(nb, a, x, lam, r, fa);
    orc_kinetic(nb, a, x, T);
#pragma omp parallel for schedule(static) collapse(2)
    for (int q = 0; q < nrhs; ++q)
        for (int c = 0; c < nch; ++c)
            for (int i = 0; i < nb; ++i) {
                size_t row = (size_t)c * nb + i;
                const zc *xq = X + (size_t)q * N;
                ld sr, si;
                if (Bx) { sr = creal(Bx[(size_t)q * N + row]); si = cimag(Bx[(size_t)q * N + row]); }
                else { sr = (c == q) ? (ld)fa[i] : 0.0L; si = 0.0L; }
                for (int j = 0; j < nb; ++j) {
                    ld t = (ld)h2m * (ld)T[(size_t)j * nb + i];
                    /* the matrix entry is the DOUBLE h2m*T_ij; use exactly that value */
                    t = (ld)(double)t;
                    if (j == i) continue;
                    sr -= t * creal(xq[(size_t)c * nb + j]);
                    si -= t * cimag(xq[(size_t)c * nb + j]);
                }
                {   /* diagonal entry exactly as assembled (step 3 evaluation order) */
                    volatile double kt = h2m * T[(size_t)i * nb + i];
                    double l = lval[c];
                    volatile double cf = h2m * l * (l + 1) / (r[i] * r[i]);
                    volatile double d = kt + cf;
                    volatile double de = ethr[c] - energy;
                    volatile double d2 = d + de;
                    zc dg = d2 + V[((size_t)i * nch + c) * nch + c];
                    ld dr = creal(dg), di = cimag(dg);
                    ld xr = creal(xq[row]), xi = cimag(xq[row]);
                    sr -= dr * xr - di * xi;
                    si -= dr * xi + di * xr;
                }
                for (int c2 = 0; c2 < nch; ++c2) {
                    if (c2 == c) continue;
                    zc v = V[((size_t)i * nch + c2) * nch + c];
                    ld vr = creal(v), vi = cimag(v);
                    ld xr = creal(xq[(size_t)c2 * nb + i]), xi = cimag(xq[(size_t)c2 * nb + i]);
                    sr -= vr * xr - vi * xi;
                    si -= vr * xi + vi * xr;
                }
                Rr[(size_t)q * N + row] = (double)sr + (double)si * I;
            }
    free(x); free(T);
    return 0;
}

/* Step 7 (PAPER.md:137 step 4 + BASELINE.json): R_cc' = (h2m/a) sum_i fa_i X[(c,i), c'].  nch x nch column-major. */
int orc_contract(int nch, int nb, double a, double h2m, const double *fa, const zc *X, zc *R) {
    size_t N = (size_t)nch * nb;
    for (int c2 = 0; c2 < nch; ++c2)
        for (int c1 = 0; c1 < nch; ++c1) {
            ld sr = 0, si = 0;
            for (int i = 0; i < nb; ++i) {
                zc xv = X[(size_t)c2 * N + (size_t)c1 * nb + i];
                sr += (ld)fa[i] * creal(xv);
                si += (ld)fa[i] * cimag(xv);
            }
            ld pf = (ld)h2m / (ld)a;
            R[(size_t)c2 * nch + c1] = (double)(pf * sr) + (double)(pf * si) * I;
        }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------
 * The whole chain: mesh -> T -> C -> LU -> solves -> two refinement steps with the long-double structured residual
 * (so the oracle's own error is ~1e-15, not the 1e-11..1e-10 a bare FP64 LU gives on this ill-conditioned C) -> R.
 * mode 0 = long-double accumulation everywhere; mode 1 = double accumulation in the O(N^3) factorisation and the
 * substitutions ("big-N mode"), residuals still long double.  X_out (N x nch) may be NULL.
 * seconds_out (may be NULL): wall time of factor + solve + refine + contract (assembly excluded).
 * ---------------------------------------------------------------------------------------------------------- */
int orc_rmatrix(int nch, int nb, double a, double h2m, const int *lval, const double *ethr, double energy,
                const zc *V, int mode, int nrefine, zc *R, zc *X_out, double *seconds_out) {
    if (nch < 1 || nb < 1) return -1;
    size_t N = (size_t)nch * nb;
    double *x = malloc(sizeof(double) * nb * 4), *lam = x + nb, *r = x + 2 * nb, *fa = x + 3 * nb;
    zc *C = malloc(sizeof(zc) * N * N);
    zc *X = malloc(sizeof(zc) * N * nch), *Rr = malloc(sizeof(zc) * N * nch);
    orc_lu f;
    if (!x || !C || !X || !Rr || lu_alloc(&f, N)) return -2;
    orc_mesh(nb, a, x, lam, r, fa);
    orc_assemble(nch, nb, a, h2m, lval, ethr, energy, V, C);
    for (size_t i = 0; i < N; ++i)
        for (size_t j = 0; j < N; ++j) f.W[i * N + j] = C[j * N + i];
    free(C);
#ifdef _OPENMP
    double t0 = omp_get_wtime();
#endif
    int info = lu_factor(&f, mode);
    if (!info) {
        orc_rhs(nch, nb, fa, X);
        lu_solve(&f, X, nch, mode);
        for (int it = 0; it < nrefine; ++it) {
            orc_structured_residual(nch, nb, a, h2m, lval, ethr, energy, V, nch, NULL, X, Rr);
            lu_solve(&f, Rr, nch, mode);
            for (size_t k = 0; k < N * nch; ++k) X[k] += Rr[k];
        }
        orc_contract(nch, nb, a, h2m, fa, X, R);
        if (X_out) memcpy(X_out, X, sizeof(zc) * N * nch);
    }
#ifdef _OPENMP
    if (seconds_out) *seconds_out = omp_get_wtime() - t0;
#else
    if (seconds_out) *seconds_out = 0;
#endif
    lu_free(&f); free(x); free(X); free(Rr);
    return info;
}
