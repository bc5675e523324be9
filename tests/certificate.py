"""A-posteriori certificate of a computed R-matrix, evaluated by the ORACLE only (test infrastructure).

C - E I is complex symmetric (symmetric kinetic + Bloch blocks, mesh-diagonal symmetric couplings), so with
X = C^-1 B exact and r = B - C X~ the residual of a computed X~,

    R_exact - R~ = (h2m/a) B^T C^-1 r = (h2m/a) X^T r = (h2m/a) X~^T r  +  (h2m/a) e^T r,     e = C^-1 r = X - X~.

The first term is computed exactly enough from the oracle's long-double matrix-free residual (oracle.structured_residual);
the second ("second-order") term is O(||C^-1|| ||r||^2).  It is bounded here by things the library did not report itself:
  * backward_err: the oracle's r in the backward-error measure of the north-star (bar: 50 N 2^-53), per right-hand side
    ||r_j||_inf / (||C||_inf ||x~_j||_inf + ||b_j||_inf), with ||C||_inf formed from the oracle's own tables (oracle.mesh /
    oracle.kinetic) and the input potential;
  * second: an explicit estimate of (h2m/a) e^T r with e from block-Jacobi steps e <- e + K_d^-1 (r - C e), K_d the Nc
    diagonal blocks (numpy LAPACK per block), C e by the oracle's matrix-free operator.  The iteration converges for the
    configs' couplings (its contraction is returned); the estimate only has to be right to a factor.
"""
import numpy as np

import oracle


def matrix_tables(w, energy):
    """(T [nb x nb, units h2m = 1], diag [nch, nb] = h2m T_ii + h2m l(l+1)/r_i^2 + E_c - E, r, fa) from the oracle."""
    x, _, r, fa = oracle.mesh(w.nb, w.a)
    T = oracle.kinetic(w.nb, w.a, x)
    l = np.asarray(w.lval, dtype=np.float64)
    diag = (w.h2m * np.diag(T))[None, :] + w.h2m * (l * (l + 1))[:, None] / (r * r)[None, :] + \
        (np.asarray(w.ethr)[:, None] - float(energy))
    return T, diag, r, fa


def anorm_inf(w, energy, V):
    """||C - E I||_inf from the block structure (Eqs. 3-4): row (c, i) holds h2m T_ij (j != i), its diagonal entry, and
    V_cc'(r_i) for c' != c.  V[i, c2, c1] = V_{c1 c2}(r_i)."""
    T, diag, _, _ = matrix_tables(w, energy)
    offT = w.h2m * (np.abs(T).sum(axis=1) - np.abs(np.diag(T)))                   # [i]
    idx = np.arange(w.nch)
    Vd = V[:, idx, idx].T                                                          # [c, i]
    coup = np.abs(V).sum(axis=1).T - np.abs(Vd)                                    # [c1, i]: sum over c2 != c1
    rows = offT[None, :] + np.abs(diag + Vd) + coup
    return float(rows.max())


def _block_solve(w, energy, V, T, diag, Z):
    """K_d^-1 Z, K_c = h2m T + diag(diag_c + V_cc)."""
    out = np.empty_like(Z)
    idx = np.arange(w.nb)
    for c in range(w.nch):
        K = (w.h2m * T).astype(np.complex128)
        K[idx, idx] = diag[c] + V[:, c, c]
        out[c * w.nb:(c + 1) * w.nb] = np.linalg.solve(K, Z[c * w.nb:(c + 1) * w.nb])
    return out


def certificate(w, energy, X, R, jacobi_steps=1):
    """X: N x nch computed solution, R: nch x nch computed R-matrix (R[c1, c2]).  Returns a dict:
    est (first-order term / max|R|), rmax (max|r|), backward_err (of the oracle's r, reading R8), second (second-order
    term / max|R|), contraction (of the last block-Jacobi step)."""
    energy = float(energy)
    T, diag, r_mesh, fa = matrix_tables(w, energy)
    V = w.potential(r_mesh)
    args = (w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, energy, V)
    res = oracle.structured_residual(*args, X)
    scale = np.abs(R).max()
    est = np.abs((w.h2m / w.a) * (X.T @ res)).max() / scale
    # backward error of reading R8, per right-hand side j: ||r_j||_inf / (||C||_inf ||x_j||_inf + ||b_j||_inf), oracle's r
    berr = (np.abs(res).max(axis=0) / (anorm_inf(w, energy, V) * np.abs(X).max(axis=0) + np.abs(fa).max())).max()
    e = _block_solve(w, energy, V, T, diag, res)
    contraction = 0.0
    for _ in range(jacobi_steps):
        rho = oracle.structured_residual(*args, e, B=res)                          # r - C e
        d = _block_solve(w, energy, V, T, diag, rho)
        contraction = np.abs(d).max() / max(np.abs(e).max(), 1e-300)
        e = e + d
    second = np.abs((w.h2m / w.a) * (e.T @ res)).max() / scale
    return {"est": float(est), "rmax": float(np.abs(res).max()), "backward_err": float(berr), "second": float(second),
            "contraction": float(contraction)}
