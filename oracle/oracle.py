"""ctypes binding of oracle/hprmat_oracle.c (numpy in, numpy out).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Every function cites the passage of /root/reference/PAPER.md it follows in hprmat_oracle.c.  Arrays are column-major
(Fortran order) complex128 unless stated.  V has shape (nb, nch, nch) C-order with V[i, c2, c1] = V_{c1 c2}(r_i).

Beside the bindings, three functions are written here in plain numpy / scipy / mpmath on top of them: collision_matrix
(matching at the channel radius, neutral and charged), rmatrix_nonlocal (full potential blocks) and the channel-function
helper _coulomb_channel.  All functions are pinned in tests/test_oracle_pins.py (list in DESIGN.md section 5.1); none is
"parity unpinned".
"""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def _L():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(_L().orc_num_threads())


def mesh(nb: int, a: float):
    """Gauss-Legendre mesh on (0,a).  Returns x (on (0,1), ascending), lam (weights on (0,1)),
    r = a*x, fa = f_i(a) (the paper's q2(r_i))."""
    x, lam, r, fa = (np.zeros(nb) for _ in range(4))
    rc = _L().orc_mesh(C.c_int(nb), C.c_double(a), _p(x), _p(lam), _p(r), _p(fa))
    if rc:
        raise ValueError(f"orc_mesh rc={rc}")
    return x, lam, r, fa


def kinetic(nb: int, a: float, x: np.ndarray) -> np.ndarray:
    """kinetic + Bloch matrix T (nb x nb, units hbar^2/2mu = 1)."""
    T = np.zeros((nb, nb), order="F")
    rc = _L().orc_kinetic(C.c_int(nb), C.c_double(a), _p(np.ascontiguousarray(x)), _p(T))
    if rc:
        raise ValueError(f"orc_kinetic rc={rc}")
    return T


def _chan(lval, ethr):
    lv = np.ascontiguousarray(lval, dtype=np.int32)
    et = np.ascontiguousarray(ethr, dtype=np.float64)
    return lv, et


def assemble(nch, nb, a, h2m, lval, ethr, energy, V) -> np.ndarray:
    """PAPER.md:87-99 Eqs. (3),(4) with Eq. (1)'s diagonal terms -- C - E*I, N x N column-major."""
    lv, et = _chan(lval, ethr)
    V = np.ascontiguousarray(V, dtype=np.complex128)
    assert V.shape == (nb, nch, nch)
    N = nch * nb
    Cm = np.zeros((N, N), dtype=np.complex128, order="F")
    rc = _L().orc_assemble(C.c_int(nch), C.c_int(nb), C.c_double(a), C.c_double(h2m), _p(lv), _p(et),
                           C.c_double(energy), _p(V), _p(Cm))
    if rc:
        raise ValueError(f"orc_assemble rc={rc}")
    return Cm


def rhs(nch, nb, fa) -> np.ndarray:
    """B[(c,i), c'] = fa_i delta_cc'."""
    N = nch * nb
    B = np.zeros((N, nch), dtype=np.complex128, order="F")
    _L().orc_rhs(C.c_int(nch), C.c_int(nb), _p(np.ascontiguousarray(fa)), _p(B))
    return B


def solve(A, B, mode: int = 0, nrefine: int = 2, return_ipiv: bool = False):
    """PAPER.md:125-137 Eq. (5) -- dense A X = B by Crout LU with partial pivoting, accumulated dot products."""
    A = np.asfortranarray(A, dtype=np.complex128)
    B = np.asfortranarray(B, dtype=np.complex128)
    if B.ndim == 1:
        B = B.reshape(-1, 1, order="F")
    n, nrhs = A.shape[0], B.shape[1]
    assert A.shape == (n, n) and B.shape[0] == n
    X = np.zeros((n, nrhs), dtype=np.complex128, order="F")
    ipiv = np.zeros(max(n, 1), dtype=np.int32)
    rc = _L().orc_solve(C.c_int(n), C.c_int(nrhs), _p(A), _p(B), _p(X), _p(ipiv), C.c_int(mode), C.c_int(nrefine))
    if rc < 0:
        raise ValueError(f"orc_solve rc={rc}")
    if rc > 0:
        raise ZeroDivisionError(f"orc_solve: zero pivot at step {rc}")
    return (X, ipiv[:n]) if return_ipiv else X


def structured_residual(nch, nb, a, h2m, lval, ethr, energy, V, X, B=None) -> np.ndarray:
    """B - (C - E I) X in long double from the block structure of Eqs. (3),(4)."""
    lv, et = _chan(lval, ethr)
    V = np.ascontiguousarray(V, dtype=np.complex128)
    X = np.asfortranarray(X, dtype=np.complex128)
    N = nch * nb
    nrhs = X.shape[1]
    assert X.shape[0] == N
    Bp = None
    if B is not None:
        B = np.asfortranarray(B, dtype=np.complex128)
        assert B.shape == X.shape
        Bp = _p(B)
    Rr = np.zeros((N, nrhs), dtype=np.complex128, order="F")
    rc = _L().orc_structured_residual(C.c_int(nch), C.c_int(nb), C.c_double(a), C.c_double(h2m), _p(lv), _p(et),
                                      C.c_double(energy), _p(V), C.c_int(nrhs), Bp, _p(X), _p(Rr))
    if rc:
        raise ValueError(f"orc_structured_residual rc={rc}")
    return Rr


def contract(nch, nb, a, h2m, fa, X) -> np.ndarray:
    """PAPER.md:137 step 4 (+ BASELINE.json prefactor) -- R = (h2m/a) B^T X."""
    X = np.asfortranarray(X, dtype=np.complex128)
    R = np.zeros((nch, nch), dtype=np.complex128, order="F")
    _L().orc_contract(C.c_int(nch), C.c_int(nb), C.c_double(a), C.c_double(h2m), _p(np.ascontiguousarray(fa)),
                      _p(X), _p(R))
    return R


def rmatrix(nch, nb, a, h2m, lval, ethr, energy, V, mode: int = 0, nrefine: int = 2, return_x=False,
            return_seconds=False):
    """Whole chain: mesh -> T -> C - E I -> LU -> solves -> refinement -> R."""
    lv, et = _chan(lval, ethr)
    V = np.ascontiguousarray(V, dtype=np.complex128)
    assert V.shape == (nb, nch, nch)
    N = nch * nb
    R = np.zeros((nch, nch), dtype=np.complex128, order="F")
    X = np.zeros((N, nch), dtype=np.complex128, order="F")
    sec = C.c_double(0.0)
    rc = _L().orc_rmatrix(C.c_int(nch), C.c_int(nb), C.c_double(a), C.c_double(h2m), _p(lv), _p(et),
                          C.c_double(energy), _p(V), C.c_int(mode), C.c_int(nrefine), _p(R), _p(X), C.byref(sec))
    if rc < 0:
        raise ValueError(f"orc_rmatrix rc={rc}")
    if rc > 0:
        raise ZeroDivisionError(f"orc_rmatrix: zero pivot at step {rc}")
    out = [R]
    if return_x:
        out.append(X)
    if return_seconds:
        out.append(sec.value)
    return out[0] if len(out) == 1 else tuple(out)


def rmatrix_nonlocal(nch, nb, a, h2m, lval, ethr, energy, W, return_x=False):
    """R-matrix with NON-LOCAL potentials ("all blocks are full matrices").

    W: N x N complex, index (c*nb + i) as everywhere: W[(c,i),(c',j)] = <f_i| W_cc' |f_j>, the matrix elements of the
    potential in the Lagrange basis, MeV (for a kernel W_cc'(r,r') at the Gauss approximation of the Lagrange-mesh method:
    a sqrt(lam_i lam_j) W_cc'(r_i, r_j); for a local potential V_cc'(r_i) delta_ij).  The matrix is Eq. (3)'s with the
    potential blocks replaced by W:  C - E I = [kinetic + Bloch + centrifugal + threshold - E on the diagonal blocks] + W;
    then Eq. (5), the Nc solves and the contraction exactly as in rmatrix() -- built from the same pinned pieces."""
    N = nch * nb
    W = np.asarray(W, dtype=np.complex128)
    assert W.shape == (N, N)
    x, lam, r, fa = mesh(nb, a)
    C0 = assemble(nch, nb, a, h2m, lval, ethr, energy, np.zeros((nb, nch, nch), dtype=np.complex128))
    X = solve(C0 + W, rhs(nch, nb, fa))
    R = contract(nch, nb, a, h2m, fa, X)
    return (R, X) if return_x else R


def _coulomb_channel(l, eta, x, is_open):
    """(F, x dF/dx, G, x dG/dx) of an open channel -- Coulomb wave functions F_l(eta, x), G_l(eta, x) -- or
    (0, 0, 1, x W'/W) of a closed one, W = W_{-eta, l+1/2}(2x) the decaying Whittaker function (only its logarithmic
    derivative matters: a column scale of Z^O drops out of the open rows).  mpmath at 30 digits; derivatives of F and G
    from the textbook recurrence  u_l' = S_{l+1} u_l - R_{l+1} u_{l+1},  S_l = l/x + eta/l,  R_l = sqrt(1 + eta^2/l^2)
    (Abramowitz & Stegun 14.2.2), the derivative of W numerically (mp.diff)."""
    import mpmath as mp
    with mp.workdps(30):
        xm, em = mp.mpf(float(x)), mp.mpf(float(eta))
        if is_open:
            S = (l + 1) / xm + em / (l + 1)
            Rr = mp.sqrt(1 + (em / (l + 1)) ** 2)
            F, F1 = mp.coulombf(l, em, xm), mp.coulombf(l + 1, em, xm)
            G, G1 = mp.coulombg(l, em, xm), mp.coulombg(l + 1, em, xm)
            return float(F), float(xm * (S * F - Rr * F1)), float(G), float(xm * (S * G - Rr * G1))
        W = mp.whitw(-em, l + mp.mpf(1) / 2, 2 * xm)
        dW = mp.diff(lambda t: mp.whitw(-em, l + mp.mpf(1) / 2, 2 * t), xm)
        return 0.0, 0.0, 1.0, float(xm * dW / W)


def collision_matrix(R, lval, ethr, energy, h2m, a, zze2=None):
    """Collision (S) matrix of the OPEN channels from the R-matrix at the channel radius.

    zze2: None (neutral case, eta = 0) or the per-channel products Z1 Z2 e^2 (MeV fm); then the Sommerfeld parameter of
    channel c is eta_c = zze2_c / (2 h2m k_c) and F, G are the Coulomb wave functions, W the Whittaker function (below).

    PAPER.md:35, 53, 71 name the step ("matching to asymptotic solutions", "collision matrix") without printing it; the
    reading taken (R14) is the standard one of the paper's ref. [2] (Descouvemont & Baye 2010):
        Z^O_cc' = (k_c' a)^-1/2 [ O_c(k_c a) delta_cc' - a R_cc' dO_c'/dr (a) ],      Z^I likewise with I,
        U = open rows of (Z^O)^-1 Z^I   (columns: open channels only),
    evaluated with I = O - 2iF substituted, Z^I = Z^O - 2i Z^F, i.e. U = 1 - 2i (Z^O)^-1 Z^F: the same matrix, but a
    channel far below its centrifugal barrier (G/F ~ 1e30) no longer loses F against G in the difference of two
    nearly equal columns (the literal form is what tests/scatter.smatrix evaluates; the two are compared in the pins).
    with k_c = sqrt(|E - E_c| / h2m); open channels: O = G + iF, I = G - iF, F = x j_l(x), G = -x y_l(x), x = k r;
    closed channels (E < E_c) carry no incoming wave and their outgoing function is the decaying one, the eta = 0
    Whittaker function W(r) = x k_l(x), x = kappa r (modified spherical Bessel function of the second kind).
    Returns (U, open) with U nopen x nopen and `open` the indices of the open channels.  Plain numpy / scipy.special
    (neutral case) or mpmath (charged case) for the channel functions.
    """
    from scipy.special import spherical_jn, spherical_yn, spherical_kn
    R = np.asarray(R, dtype=np.complex128)
    nch = R.shape[0]
    ekin = float(energy) - np.asarray(ethr, dtype=float)
    x = np.sqrt(np.abs(ekin) / h2m) * a
    O = np.zeros(nch, dtype=complex)
    dO = np.zeros(nch, dtype=complex)   # x * dO/dx = a * dO/dr at r = a
    Fr = np.zeros(nch)
    dFr = np.zeros(nch)                 # x * dF/dx
    charged = zze2 is not None and np.any(np.asarray(zze2, dtype=float) != 0.0)
    for c in range(nch):
        l, xc = int(lval[c]), x[c]
        if charged:
            eta = float(zze2[c]) / (2.0 * h2m * (xc / a))
            F, xdF, G, xdG = _coulomb_channel(l, eta, xc, ekin[c] > 0)
            O[c], dO[c] = G + 1j * F, xdG + 1j * xdF
            Fr[c], dFr[c] = F, xdF
        elif ekin[c] > 0:
            F = xc * spherical_jn(l, xc)
            dF = spherical_jn(l, xc) + xc * spherical_jn(l, xc, derivative=True)
            G = -xc * spherical_yn(l, xc)
            dG = -spherical_yn(l, xc) - xc * spherical_yn(l, xc, derivative=True)
            O[c], dO[c] = G + 1j * F, xc * (dG + 1j * dF)
            Fr[c], dFr[c] = F, xc * dF
        else:
            W = xc * spherical_kn(l, xc)
            dW = spherical_kn(l, xc) + xc * spherical_kn(l, xc, derivative=True)
            O[c], dO[c] = W, xc * dW
    opn = np.nonzero(ekin > 0)[0]
    ZO = (np.diag(O) - R * dO[None, :]) / np.sqrt(x)[None, :]
    ZF = ((np.diag(Fr) - R * dFr[None, :]) / np.sqrt(x)[None, :])[:, opn]
    Y = np.linalg.solve(ZO, ZF)
    return np.eye(len(opn)) - 2j * Y[opn, :], opn


# ---- propagation over sub-intervals ("propagation", ns sub-intervals; reading R16) ----------
def sector_tables(nb: int, a_lo: float, a_hi: float):
    """Lagrange-Legendre mesh on the sub-interval (a_lo, a_hi), NOT regularised, with the definitions written out:
    f_i(r) = l_i(x) / sqrt(h lam_i), x = (r - a_lo)/h, l_i(x) = prod_{m != i} (x - x_m)/(x_i - x_m).  Returns
    (r, fa_left, fa_right, T) with T_ij = <f_i| -d2/dr2 + L(a_hi) - L(a_lo) |f_j> = int f_i' f_j' dr (Bloch operator at both
    ends; units hbar^2/2mu = 1), the integral by the mesh's own Gauss quadrature, exact for this polynomial integrand.
    l_i'(x_k) from the product rule: for k != i only the term without the factor (x - x_k) survives,
    l_i'(x_k) = prod_{m != i,k} (x_k - x_m) / prod_{m != i} (x_i - x_m);  l_i'(x_i) = sum_{m != i} 1/(x_i - x_m).
    long double throughout, rounded to double at the end."""
    x, lam, _, _ = mesh(nb, 1.0)
    xl = x.astype(np.longdouble)
    ll = lam.astype(np.longdouble)
    h = np.longdouble(a_hi) - np.longdouble(a_lo)
    D = np.zeros((nb, nb), dtype=np.longdouble)          # D[k, i] = l_i'(x_k)
    l0 = np.zeros(nb, dtype=np.longdouble)
    l1 = np.zeros(nb, dtype=np.longdouble)
    for i in range(nb):
        others = [m for m in range(nb) if m != i]
        den = np.prod(xl[i] - xl[others])
        l0[i] = np.prod(0 - xl[others]) / den
        l1[i] = np.prod(1 - xl[others]) / den
        D[i, i] = np.sum(1 / (xl[i] - xl[others]))
        for k in others:
            rest = [m for m in others if m != k]
            D[k, i] = np.prod(xl[k] - xl[rest]) / den
    T = np.zeros((nb, nb), dtype=np.longdouble)
    for i in range(nb):
        for j in range(nb):
            T[i, j] = np.sum(ll * D[:, i] * D[:, j]) / (h * h * np.sqrt(ll[i] * ll[j]))
    r = (np.longdouble(a_lo) + h * xl).astype(np.float64)
    return r, (l0 / np.sqrt(h * ll)).astype(np.float64), (l1 / np.sqrt(h * ll)).astype(np.float64), T.astype(np.float64)


def sector_matrices(nch, nb, a_lo, a_hi, h2m, lval, ethr, energy, V):
    """Rsec_ab = h2m B_a^T (C - E I)^-1 B_b for a, b in {L, R} on the sub-interval (a_lo, a_hi): returns the 2 x 2 nested list
    [[LL, LR], [RL, RR]] of nch x nch matrices.  C - E I has the structure of Eqs. (3),(4) with the sector's T; dense
    assembly, the oracle's LU (orc_solve) for the 2 nch right-hand sides."""
    r, faL, faR, T = sector_tables(nb, a_lo, a_hi)
    V = np.asarray(V, dtype=np.complex128)
    assert V.shape == (nb, nch, nch)
    N = nch * nb
    Cm = np.zeros((N, N), dtype=np.complex128)
    for c in range(nch):
        blk = (h2m * T).astype(np.complex128)
        blk[np.arange(nb), np.arange(nb)] += h2m * lval[c] * (lval[c] + 1) / r ** 2 + (ethr[c] - energy)
        Cm[c * nb:(c + 1) * nb, c * nb:(c + 1) * nb] = blk
    for i in range(nb):
        idx = np.arange(nch) * nb + i
        Cm[np.ix_(idx, idx)] += V[i].T                      # V[i, c2, c1] = V_{c1 c2}(r_i)
    B = np.zeros((N, 2 * nch), dtype=np.complex128)
    for c in range(nch):
        B[c * nb:(c + 1) * nb, c] = faL
        B[c * nb:(c + 1) * nb, nch + c] = faR
    X = solve(Cm, B)
    G = h2m * (B.T @ X)
    return [[G[:nch, :nch], G[:nch, nch:]], [G[nch:, :nch], G[nch:, nch:]]]


def propagate(a_lo, a_hi, R_in, Rsec):
    """a_hi R_out = Rsec_RR - Rsec_RL (Rsec_LL + a_lo R_in)^-1 Rsec_LR  (reading R16: u(a_hi) = Rsec_RR u'(a_hi) - Rsec_RL u'(a_lo),
    u(a_lo) = Rsec_LR u'(a_hi) - Rsec_LL u'(a_lo), u(a_lo) = a_lo R_in u'(a_lo); eliminate u'(a_lo))."""
    (LL, LR), (RL, RR) = Rsec
    return (RR - RL @ np.linalg.solve(LL + a_lo * np.asarray(R_in), LR)) / a_hi
