// refine.cuh -- the stopping rule of the iterative refinement ("checks convergence (maximum residual
// modulus)", no threshold given, reading R9), shared by the structured and the raw mixed solves.
#pragma once

namespace hp {

// dn = max|d_k|, xn = max|X|, dprev = max|d_{k-1}| (k = 1: max|X_0|).  The error left after this step is estimated as
// dn * rho / (1 - rho) with the observed contraction rho = dn / dprev.
enum { REF_CONTINUE = 0, REF_CONVERGED = 1, REF_STAGNATED = 2 };
inline int refine_verdict(double dn, double xn, double dprev, double tol) {
    if (!(dn == dn) || !(xn == xn)) return REF_STAGNATED;  // NaN
    if (dn <= tol * xn * 1e-3) return REF_CONVERGED;        // correction already far below the target
    const double rho = dprev > 0.0 ? dn / dprev : 1.0;
    if (rho >= 0.5) return REF_STAGNATED;
    if (dn * rho / (1.0 - rho) <= tol * xn) return REF_CONVERGED;
    return REF_CONTINUE;
}

}  // namespace hp
