/*
 * hprmat.h -- C ABI of the B200-native (sm_100a) hot path of the R-matrix method of arxiv 2512.11590 (HPRMAT).
 *
 * What the library computes (citations are /root/reference/PAPER.md lines):
 *   - the dense complex-symmetric Lagrange-Legendre internal-region matrix  C - E*I  of Eqs. (1),(3),(4)
 *     (PAPER.md:73-99), N = nch*nbasis, row/column index of (channel c, mesh point i) = c*nbasis + i;
 *   - the solution X of (C - E*I) X = B for the nch right-hand sides B[(c,i),c'] = f_i(a) delta_cc'
 *      by blocked LU with partial pivoting, M = P L U (Eq. 5), either in
 *     FP64 (the paper's Type 1) or with low-precision factors plus FP64 iterative refinement (Types 2/4,
 *     PAPER.md:147-151, 192-230), the low-precision factorisation being applied to the block-diagonally
 *     preconditioned matrix K_diag^-1 M of the paper's Type 3 (Eqs. 7-9);
 *   - the R-matrix  R_cc' = (hbar^2/2 mu a) sum_i f_i(a) X[(c,i),c']  (PAPER.md:137 step 4; prefactor from
 *     BASELINE.json north_star).
 *
 * Conventions
 *   - All matrices are COLUMN-MAJOR.  "complex" is interleaved (re, im) double unless stated.
 *   - Pointers marked  dev  are CUDA device pointers, those marked  host  are host pointers.  The library never
 *     allocates device memory inside hprmat_solve / hprmat_zsolve / hprmat_zgetrf / hprmat_zgetrs / hprmat_zgemm.
 *   - Every call enqueues its kernels on the stream given at setup (or as argument); calls that fill a host
 *     hprmat_info synchronise that stream ONCE, at the end, to read the device-side status (the stopping rule of the
 *     refinement is evaluated on the device after every step); calls with info == NULL never synchronise -- their status
 *     stays on the device and is fetched with hprmat_last_status.
 *     Part of a factorisation (the kept block inverses) runs on a side stream owned by the context (by the library, per
 *     device, for the raw entries), joined before the call's work on the caller's stream continues.
 *   - Return value: 0 success; -k = argument k (1-based) invalid; >0 = one of the HPRMAT_E* codes below.
 *   - There is NO CPU fallback: without a CUDA device every compute entry returns HPRMAT_ECUDA.
 *   - One context per host thread / stream; different contexts may be used concurrently from different host threads
 *     (algorithm switches, side streams and status words are per context; the only process-wide state are the defaults
 *     hprmat_fp64_algo / hprmat_zgemm_algo, the launch counter and the optional profile record of hprmat_profile.h).
 *     The caller owns V, R, A, B, ipiv and the workspace; the context owns everything else and is reused across an
 *     energy scan.
 */
#ifndef HPRMAT_H
#define HPRMAT_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hprmat_ctx hprmat_ctx; /* opaque */

/* precision modes (PAPER.md:253-269 solver_type; Fig. 3) */
enum {
    HPRMAT_FP64 = 1,         /* FP64 LU of C - E*I on FP64 tensor cores (+ refinement with a compensated residual)     */
    HPRMAT_MIXED = 2,        /* low-precision (complex64 storage, TF32 tensor-core update) LU, NO refinement            */
    HPRMAT_MIXED_REFINE = 3, /* low-precision LU + FP64 residual / iterative refinement to double accuracy            */
    HPRMAT_TYPE3 = 4         /* the paper's Type 3 as printed (Eqs. 7-9; local potentials only): the     */
                             /* point-major Schur matrix I + K^-1 V with the REAL kinetic block K shared by all channels   */
                             /* (its inverse and K^-1 q2 are energy-independent: computed once at hprmat_setup and reused   */
                             /* across the scan), complex64 LU with partial pivoting and FP32-class (3xTF32) products, no   */
                             /* refinement: ~1e-6 in R, the accuracy the paper quotes for Type 3             */
};

/* status codes */
enum {
    HPRMAT_OK = 0,
    HPRMAT_ESINGULAR = 1,     /* exact zero pivot; info->pivot_index = 1-based column                                  */
    HPRMAT_ENOTCONVERGED = 2, /* refinement hit max_refine or stagnated; X / R hold the last iterate    */
    HPRMAT_ENOMEM = 3,        /* device allocation failed at setup, or workspace too small                             */
    HPRMAT_ECUDA = 4,         /* CUDA error (no device, launch failure, ...); see hprmat_last_cuda_error()             */
    HPRMAT_EUNVERIFIED = 5    /* hprmat_last_status only: the factorisation with verified diagonal pivots of an          */
                              /* UNSYNCHRONISED call was refuted (or its preconditioner is singular / ill-conditioned at */
                              /* this energy); X / R are not certified -- repeat the call with info != NULL, which falls  */
                              /* back to the pivoting factorisation by itself                                            */
};

typedef struct {
    int status;            /* same as the return value                                                                  */
    int refine_steps;      /* refinement steps actually taken                                                           */
    int pivot_index;       /* first zero pivot (1-based) or 0                                                           */
    int reserved;          /* block panels whose diagonal-pivot speculation was refuted in the first attempt (the call   */
                           /* then refactored with pivoting); 0 in the normal case                                       */
    double resid_max;      /* max_ij |B - A X|_ij of the last residual evaluated (absolute)                             */
    double backward_err;   /* max_j ||b_j - A x_j||_inf / (||A||_inf ||x_j||_inf + ||b_j||_inf); <0 if not evaluated     */
    double ms_assemble, ms_lu, ms_solve, ms_refine, ms_contract, ms_total; /* CUDA-event stage times, milliseconds      */
    double lu_tflops;      /* (8 N^3 / 3) / ms_lu, the paper's flop convention                           */
} hprmat_info;

/* ---- structured R-matrix path ------------------------------------------------------------------------------------ */

/* Create a context for nch channels and nbasis Lagrange-Legendre functions on (0, a).
 *   a      channel radius, fm;  h2m = hbar^2/2mu, MeV fm^2 (equal reduced mass in all channels)
 *   lval   host, int[nch]: orbital momenta l_c;  ethr  host, double[nch]: thresholds E_c, MeV (enter as +E_c on the
 *          diagonal of Eq. 1)
 *   max_mode  bitwise OR of (1 << HPRMAT_FP64), (1 << HPRMAT_MIXED), (1 << HPRMAT_MIXED_REFINE), (1 << HPRMAT_TYPE3): sizes the buffers
 *          (FP64: 16 N^2 bytes; mixed: 8 N^2 bytes; plus O(N nch)).  0 means all modes.
 *   cuda_stream  a cudaStream_t (may be NULL = default stream)
 * Computes the mesh, f_i(a) and the kinetic + Bloch table on the host in long double and uploads them. */
int hprmat_setup(hprmat_ctx **out, int nch, int nbasis, double a, double h2m, const int *lval, const double *ethr,
                 int max_mode, void *cuda_stream);

/* Mesh abscissas r_i = a x_i (ascending, fm) and surface values f_i(a) (the paper's q2(r_i)) so the
 * caller can evaluate V_cc'(r_i).  r, fa: host, double[nbasis]; either may be NULL. */
int hprmat_mesh(const hprmat_ctx *ctx, double *r, double *fa);

/* One energy point: assemble, factorise, solve, (refine), contract.
 *   V    dev, complex [nbasis][nch][nch]: V[(i*nch + c2)*nch + c1] = V_{c1 c2}(r_i), MeV (Eq. 4)
 *   mode one of HPRMAT_FP64 / HPRMAT_MIXED / HPRMAT_MIXED_REFINE / HPRMAT_TYPE3 (must be inside max_mode)
 *   max_refine  maximum refinement steps; <0 = default (2 for FP64, 5 for MIXED_REFINE)
 *   tol  refinement stops when the estimated relative error left in X (correction norm x observed contraction, DESIGN.md
 *        reading R9) is <= tol; <=0 = default: 1e-13 in FP64 mode, 1e-12 in the mixed modes
 *   R    dev, complex nch x nch column-major (output)
 *   info host, may be NULL: then the call only enqueues work (no synchronisation in any mode): up to max_refine refinement
 *        steps in FP64 mode, one more than the previous solve needed in HPRMAT_MIXED_REFINE; the device-side stopping rule
 *        turns the steps after convergence into no-ops, and hprmat_last_status reports the outcome.
 *        With info the call enqueues as many steps as the previous solve of this context in this mode needed, reads the
 *        device status once, and continues step by step only if the stopping rule has not fired yet. */
int hprmat_solve(hprmat_ctx *ctx, double energy, const void *V, int mode, int max_refine, double tol, void *R,
                 hprmat_info *info);

/* What the FP64 LU of hprmat_solve(HPRMAT_FP64) is applied to:
 *   1 = C - E I itself (the paper's Type 1: ZGESV semantics on the assembled matrix);
 *   2 = S = K_d^-1 (C - E I), K_d = the nch diagonal blocks inverted in FP64 (the matrix of the paper's Type 3, Eqs. 7-9, here
 *       in FP64): the same N x N LU with partial pivoting and 8N^3/3 flops, but the pivots are the diagonal ones, which the
 *       panel kernel verifies instead of searching.  Default, chosen by measurement.
 * Residual, refinement and the reported backward error always refer to the original system.  A synchronised call
 * (info != NULL) falls back to variant 1 by itself when a diagonal block is singular, a multiplier refutes the diagonal
 * pivots, the correction of the refinement step stays above 1e-9 |X| or the backward error exceeds 50 N 2^-53 (E on or
 * next to a pole of an UNCOUPLED channel, possible with real potentials only); an unsynchronised call cannot, and
 * hprmat_last_status then returns HPRMAT_EUNVERIFIED.  Any other value only queries.  Returns the setting in force.
 * This is the PROCESS DEFAULT, read by every context that has no setting of its own (hprmat_set_option);
 * hprmat_solve_nonlocal follows the same switch (K_d then holds the full diagonal blocks), hprmat_zsolve / hprmat_zgetrf
 * always factor the matrix they are given. */
int hprmat_fp64_algo(int algo);

/* Per-context settings.  value 0 = follow the process default again. */
enum {
    HPRMAT_OPT_FP64_ALGO = 1,  /* 1 or 2, see hprmat_fp64_algo                                                           */
    HPRMAT_OPT_ZGEMM_ALGO = 2, /* 3 or 4, see hprmat_zgemm_algo                                                          */
    HPRMAT_OPT_GRAPHS = 3      /* 1 (default): the factorisation and every triangular solve of this context are captured    */
                               /* into CUDA graphs on first use and replayed with one launch each; 0: plain stream launches */
};
int hprmat_set_option(hprmat_ctx *ctx, int option, int value);

/* Outcome of the last hprmat_solve / hprmat_solve_nonlocal of this context -- for calls made with info == NULL, which
 * leave their status on the device.  Synchronises the context's stream, then decodes the device status words as a
 * synchronised call does: HPRMAT_OK, HPRMAT_ESINGULAR (pivot_index: 1-based column), HPRMAT_ENOTCONVERGED (mixed+refine),
 * or HPRMAT_EUNVERIFIED (see above).  refine_steps / pivot_index: host, may be NULL.  -1 if nothing was solved yet. */
int hprmat_last_status(hprmat_ctx *ctx, int *refine_steps, int *pivot_index);

/* Same call with HOST buffers (the end-to-end entry): V_host complex [nbasis][nch][nch] and R_host complex nch x nch are
 * host pointers (pinned memory makes the copies asynchronous); the host->device copy of V, all kernels and the
 * device->host copy of R are enqueued on the context's stream, which is synchronised before returning. */
int hprmat_solve_host(hprmat_ctx *ctx, double energy, const void *V_host, int mode, int max_refine, double tol,
                      void *R_host, hprmat_info *info);

/* Non-local potentials ("all blocks are full matrices"): one energy point
 * with a dense matrix of potential matrix elements instead of the mesh-diagonal V.
 *   W    dev, complex N x N column-major, leading dimension ldw >= N, N = nch*nbasis, index (c*nbasis + i):
 *        W[(c2*nbasis + j)*ldw + c1*nbasis + i] = <f_i| W_{c1 c2} |f_j>, MeV -- for a kernel W_{c1 c2}(r, r') at the Gauss
 *        approximation of the Lagrange-mesh method  a sqrt(lambda_i lambda_j) W_{c1 c2}(r_i, r_j)  (lambda: the
 *        Gauss-Legendre weights on (0,1)); a local potential is V_{c1 c2}(r_i) delta_ij.  Not modified.
 *   mode any of the three modes the context was set up with (-5 otherwise).  The mixed modes factor, in TF32,
 *        S = K_d^-1 (C - E I) with K_d the FULL diagonal blocks (kinetic terms + W_cc), inverted in FP64.
 *   max_refine, tol, R, info: as hprmat_solve.  The refinement residual B - (K + W) X is formed in working precision
 *        (W X on the FP64 tensor cores): it restores the backward error, not digits beyond kappa 2^-53.
 * The matrix is C - E I = W + [kinetic + Bloch + centrifugal + threshold - E on the diagonal blocks]; LU, solves,
 * contraction and hprmat_get_x as in hprmat_solve. */
int hprmat_solve_nonlocal(hprmat_ctx *ctx, double energy, const void *W, long ldw, int mode, int max_refine, double tol,
                          void *R, hprmat_info *info);

/* ---- propagation over sub-intervals (hprmat_init(nr, ns, rmax, zrma)) ----
 *
 * PAPER.md names the propagation and the number of sub-intervals ns without printing formulas (they are in its ref. [2]);
 * the reading taken is DESIGN.md section 3, R16.  The first sub-interval (0, a_1) is an ordinary context (hprmat_setup with
 * a = a_1, hprmat_solve -> R at a_1).  Every further sub-interval (a_lo, a_hi), a_lo > 0, gets a SECTOR context: plain
 * Lagrange-Legendre mesh on the interval, Bloch operators at both ends, the same matrix structure and the same hot path
 * (assembly, LU, solves, refinement), with two sets of nch right-hand sides -- the surface vectors of the two ends -- on one
 * factorisation.  hprmat_mesh returns the radii r_i = a_lo + (a_hi - a_lo) x_i and the RIGHT-end surface values. */
int hprmat_setup_sector(hprmat_ctx **out, int nch, int nbasis, double a_lo, double a_hi, double h2m, const int *lval,
                        const double *ethr, int max_mode, void *cuda_stream);

/* Sector matrices of one energy point:  Rsec_ab = (hbar^2/2mu) B_a^T (C - E I)^-1 B_b,  a, b in {L (= a_lo), R (= a_hi)}.
 *   V     dev, complex [nbasis][nch][nch] at the sector's mesh radii (layout as hprmat_solve)
 *   mode  HPRMAT_FP64 / HPRMAT_MIXED / HPRMAT_MIXED_REFINE;  max_refine, tol as hprmat_solve
 *   Rsec  dev, complex, four nch x nch column-major blocks in the order LL, LR, RL, RR (4 nch^2 elements)
 *   info  host, REQUIRED (the two passes are synchronised); times are summed over both passes
 * hprmat_get_x afterwards returns the solution block of the LEFT-end right-hand sides. */
int hprmat_solve_sector(hprmat_ctx *ctx, double energy, const void *V, int mode, int max_refine, double tol, void *Rsec,
                        hprmat_info *info);

/* R-matrix at a_hi from the R-matrix at a_lo and the sector matrices of (a_lo, a_hi):
 *     a_hi R_out = Rsec_RR - Rsec_RL (Rsec_LL + a_lo R_in)^-1 Rsec_LR
 * (R in this library's convention u(a) = a R u'(a), i.e. with the prefactor hbar^2/(2 mu a)).  All matrices dev, complex
 * nch x nch column-major; R_out may not alias R_in or Rsec.  info_dev: dev int[1], 0 or the 1-based zero pivot of the
 * nch x nch LU.  workspace: dev, 256-byte aligned, >= hprmat_propagate_workspace_bytes(nch).  No synchronisation. */
size_t hprmat_propagate_workspace_bytes(int nch);
int hprmat_propagate(void *cuda_stream, int nch, double a_lo, double a_hi, const void *R_in, const void *Rsec, void *R_out,
                     int *info_dev, void *workspace, size_t workspace_bytes);

/* hprmat_propagate for callers that may not allocate device memory (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same arguments, same arithmetic and same result, but the workspace is a file-scope
 * device array of the library (3 MiB, held by every GPU that loads the library until the process exits) instead of a
 * caller's buffer.  The call itself makes no cudaMalloc / cudaFree and calls no allocating routine.
 *   nch <= hprmat_propagate_static_max_nch() = 128; a larger nch returns HPRMAT_ENOMEM and hprmat_last_cuda_error() names the
 *   limit (use hprmat_propagate with a workspace then).
 * There is ONE array per device, shared by every call and cleared at the start of each: calls whose GPU work can overlap
 * (different streams, several host threads) RACE on it -- issue them on one stream, or order them with events. */
int hprmat_propagate_static_max_nch(void);
int hprmat_propagate_static(void *cuda_stream, int nch, double a_lo, double a_hi, const void *R_in, const void *Rsec,
                            void *R_out, int *info_dev);

/* Solution block of the last hprmat_solve: X dev, complex N x nch column-major (copy out). */
int hprmat_get_x(const hprmat_ctx *ctx, void *X);

/* Assembly only (Eqs. 3-4): C dev, complex N x N column-major, ldc = N. */
int hprmat_get_matrix(hprmat_ctx *ctx, double energy, const void *V, void *C);

int hprmat_destroy(hprmat_ctx *ctx);

/* ---- matching at the channel radius ------------------------------------------------- */

/* Collision matrix U of the open channels from the R-matrix: PAPER.md:35, 53, 71 name the step ("matching to asymptotic
 * solutions", "collision matrix") and defer to the paper's ref. [2]; the formula taken is DESIGN.md section 3, reading R14:
 *     Z^O_cc' = (k_c' a)^-1/2 [ O_c(a) delta_cc' - R_cc' a (dO_c'/dr)(a) ],  Z^I likewise,  U = open rows of (Z^O)^-1 Z^I,
 * with O = G + iF, I = G - iF, F and G the Coulomb wave functions F_l(eta_c, k_c r), G_l(eta_c, k_c r),
 * k_c = sqrt((E - E_c)/h2m), eta_c = zze2_c / (2 h2m k_c), in an open channel, and the decaying Whittaker function
 * W_{-eta_c, l+1/2}(2 kappa_c r), no incoming wave, in a closed one (E < E_c).
 * Evaluated as U = 1 - 2i (Z^O)^-1 Z^F (Z^I = Z^O - 2i Z^F), which stays accurate far below a barrier.
 *   nch, lval (host int[nch]), ethr (host double[nch], MeV), energy (MeV), h2m (MeV fm^2), a (fm): as in hprmat_setup
 *   zze2   host double[nch]: Z1 Z2 e^2 of each channel, MeV fm (e^2 = 1.43996 MeV fm); NULL = neutral (eta = 0)
 *   R      dev, complex nch x nch column-major: the output of hprmat_solve at this energy (not modified)
 *   U      dev, complex nopen x nopen column-major, leading dimension nopen (output); open channels keep their order
 *   nopen  host int[1] (output): number of channels with energy > ethr[c]; known when the call returns
 *   info_dev  dev int[1]: 0, or the 1-based index of a zero pivot of Z^O (U is then meaningless)
 *   workspace dev, 256-byte aligned, >= hprmat_collision_workspace_bytes(nch); owned by the caller
 * The 4 nch channel constants are computed on the host in long double (hprmat_channel_functions) and uploaded; both
 * matrices, the FP64 LU solve (hprmat_zgetrf / hprmat_zgetrs code path) and the extraction run on the stream; no
 * synchronisation.
 * Errors: negative = index of the offending argument (-6: energy equals a threshold, where k_c = 0, or lies so close to
 * one that the continued fractions of the charged channel functions do not converge), HPRMAT_ENOMEM, HPRMAT_ECUDA. */
size_t hprmat_collision_workspace_bytes(int nch);
int hprmat_collision(void *cuda_stream, int nch, const int *lval, const double *ethr, const double *zze2, double energy,
                     double h2m, double a, const void *R, void *U, int *nopen, int *info_dev, void *workspace,
                     size_t workspace_bytes);

/* Host-only helper (no CUDA call): the channel functions the matching uses, at x = k r (open) or kappa r (closed).
 *   open != 0:  out[0..3] = F_l(eta, x), x dF/dx, G_l(eta, x), x dG/dx   (Coulomb wave functions; eta = 0: x j_l, -x y_l)
 *   open == 0:  out[0..3] = 0, 0, 1, x W'/W   of W_{-eta, l+1/2}(2x)     (eta = 0: x k_l(x))
 * Long double inside (Steed's continued fractions for eta != 0, Bessel recurrences for eta = 0), rounded to double.
 * Returns 0, or minus the index of the offending argument (-3 also when x is too small for the continued fractions). */
int hprmat_channel_functions(int l, double eta, double x, int open, double *out);

/* ---- raw dense complex entries (PAPER.md:119 "take M, b, return c"; :125-137 ZGESV) -------------------------------- */

/* Workspace (bytes) needed by hprmat_zsolve / hprmat_zgetrf / hprmat_zgetrs for an n x n system with nrhs right-hand
 * sides in the given mode. */
size_t hprmat_workspace_bytes(int n, int nrhs, int mode);

/* Solve A X = B.  A dev complex n x n (lda >= n); B dev complex n x nrhs (ldb >= n), overwritten by X;
 * ipiv dev int[n], 1-based LAPACK row interchanges (of the matrix actually factorised: A itself in FP64 mode).
 * HPRMAT_FP64: A is OVERWRITTEN by its LU factors (unit-lower L and U, LAPACK zgetrf layout).
 * HPRMAT_MIXED / HPRMAT_MIXED_REFINE: A is preserved; the factors of the row/column-equilibrated complex64 copy live
 * in the workspace; refinement uses the FP64 residual B - A X and contracts by ~sqrt(n) 2^-11 kappa per
 * step (single-pass TF32 trailing update), so max_refine < 0 means 12 here; beyond kappa ~ 1e3 the call returns
 * HPRMAT_ENOTCONVERGED with the last iterate and HPRMAT_FP64 is the mode to use.
 * workspace dev, workspace_bytes >= hprmat_workspace_bytes(n, nrhs, mode). */
int hprmat_zsolve(void *cuda_stream, int n, int nrhs, void *A, int lda, void *B, int ldb, int *ipiv, int mode,
                  int max_refine, double tol, void *workspace, size_t workspace_bytes, hprmat_info *info);

/* FP64 LU with partial pivoting in place (Eq. 5): A = P L U.  info_dev: dev int[1], 0 or first zero pivot (1-based). */
int hprmat_zgetrf(void *cuda_stream, int n, void *A, int lda, int *ipiv, int *info_dev, void *workspace,
                  size_t workspace_bytes);

/* Triangular solves with the factors of hprmat_zgetrf (same workspace, untouched in between): B <- A^-1 B. */
int hprmat_zgetrs(void *cuda_stream, int n, int nrhs, const void *A, int lda, const int *ipiv, void *B, int ldb,
                  void *workspace, size_t workspace_bytes);

/* C <- beta*C + alpha*A*B, complex128 column-major, real alpha and beta; the FP64 tensor-core (DMMA) kernels that
 * perform the trailing update of the LU (3M decomposition by default, see hprmat_zgemm_algo).  A m x k, B k x n, C m x n.
 * C may alias B only when m <= 128 and beta == 0. */
int hprmat_zgemm(void *cuda_stream, int m, int n, int k, double alpha, const void *A, int lda, const void *B, int ldb,
                 double beta, void *C, int ldc);

/* Real decomposition of the complex128 product inside hprmat_zgemm and the FP64 LU: 4 = four real products per complex
 * product ("4M", componentwise accurate), 3 = three ("3M": 25 % fewer tensor-core instructions, imaginary part normwise
 * accurate; the default, chosen by measurement).  Any other value only queries.  Returns the
 * setting in force.  Process default; a context may carry its own (hprmat_set_option). */
int hprmat_zgemm_algo(int algo);

/* C <- beta*C + alpha*A*B on SPLIT-complex (planar) complex64 operands: every matrix is a pair of column-major float
 * planes (re, im).  The tcgen05 (kind::tf32, FP32 accumulation in TMEM) kernel that performs the trailing update of the
 * low-precision LU of the mixed modes.  All pointers dev; plane base addresses 16-byte
 * aligned; lda, ldb multiples of 4.  Operands are rounded to TF32 (10-bit mantissa) by the tensor core. */
int hprmat_cgemm_tf32(void *cuda_stream, int m, int n, int k, float alpha, const float *A_re, const float *A_im, int lda,
                      const float *B_re, const float *B_im, int ldb, float beta, float *C_re, float *C_im, int ldc);

/* Same operation with FP32-class accuracy ("3xTF32": every operand split in registers into two TF32 terms, three
 * mma.sync products per real product, FP32 accumulation): the GEMM of the triangular solves of the mixed modes, whose
 * O(1) right-hand sides must not be rounded to 10 mantissa bits.  Same argument rules. */
int hprmat_cgemm_3xtf32(void *cuda_stream, int m, int n, int k, float alpha, const float *A_re, const float *A_im, int lda,
                        const float *B_re, const float *B_im, int ldb, float beta, float *C_re, float *C_im, int ldc);

const char *hprmat_strerror(int code);
const char *hprmat_last_cuda_error(void);
#ifdef __cplusplus
}
#endif
#endif /* HPRMAT_H */
