// refine.cuh -- the stopping rule of the iterative refinement ("checks convergence (maximum residual
// modulus)", no threshold given, reading R9), shared by the structured and the raw mixed solves, and
// evaluated ON THE DEVICE after every step (refine_verdict_kernel, ctx.cu) so that no host round trip separates the steps.
#pragma once
#include "common.cuh"

namespace hp {

// dn = max|d_k|, xn = max|X|, dprev = max|d_{k-1}| (k = 1: max|X_0|).  The error left after this step is estimated as
// dn * rho / (1 - rho) with the observed contraction rho = dn / dprev.
enum { REF_CONTINUE = 0, REF_CONVERGED = 1, REF_STAGNATED = 2 };
__host__ __device__ inline int refine_verdict(double dn, double xn, double dprev, double tol) {
    if (!(dn == dn) || !(xn == xn)) return REF_STAGNATED;  // NaN
    if (dn <= tol * xn * 1e-3) return REF_CONVERGED;        // correction already far below the target
    const double rho = dprev > 0.0 ? dn / dprev : 1.0;
    if (rho >= 0.5) return REF_STAGNATED;
    if (dn * rho / (1.0 - rho) <= tol * xn) return REF_CONVERGED;
    return REF_CONTINUE;
}

// Device-resident state of one solve (a context's d_scal / d_info words; ctx.cu).  Doubles:
enum { SC_DN = 0, SC_XN = 1, SC_X0 = 2, SC_RMAX = 3, SC_ANORM = 4, SC_BERR = 5, SC_BNORM = 6, SC_DPREV = 8, SC_DN_LAST = 9,
       SC_XN_LAST = 10, SC_NWORDS = 16 };
// ints:
enum { IN_ZERO_PIVOT = 0, IN_KBLOCK_SINGULAR = 1, IN_VERDICT = 2, IN_STEPS = 3, IN_REFUTED = 4, IN_NWORDS = 8 };

}  // namespace hp
