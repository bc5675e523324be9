"""Pins of the CPU oracle (oracle/) against things OTHER than itself: library quadrature, exact polynomial integrals in
mpmath, Cramer's rule / Gauss-Jordan on tiny systems, closed-form R-matrices, symmetry and unitarity.
All CPU-only ("-m 'not gpu'").  Each test names the passage of PAPER.md whose step it pins.
"""
import itertools

import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_2512_11590_b200.workloads import H2M, make_workload
from scatter import R_constant_potential, smatrix

# ---------------------------------------------------------------------------------------------------- mesh


@pytest.mark.parametrize("nb", [1, 2, 5, 8, 50, 100])
def test_mesh_matches_library_gauss_legendre(nb):
    x, lam, r, fa = oracle.mesh(nb, 7.5)
    t, w = np.polynomial.legendre.leggauss(nb)
    assert np.allclose(x, (1 + t) / 2, rtol=0, atol=2e-16 * 4)
    assert np.allclose(lam, w / 2, rtol=5e-12, atol=0)   # numpy weights are plain double
    assert np.allclose(r, 7.5 * x, rtol=3e-16, atol=0)
    assert np.all(np.diff(x) > 0)
    assert np.allclose(x + x[::-1], 1.0, atol=4e-16)


@pytest.mark.parametrize("nb", [3, 10, 50])
def test_mesh_quadrature_exact_to_degree_2nb_minus_1(nb):
    x, lam, _, _ = oracle.mesh(nb, 1.0)
    assert abs(lam.sum() - 1.0) < 5e-16 * nb
    for k in range(0, 2 * nb, max(1, nb // 5)):
        assert abs(np.sum(lam * x ** k) - 1.0 / (k + 1)) < 1e-14


# ---------------------------------------------------- basis values and kinetic + Bloch table

def _lagrange_functions(nb, a, dps=50):
    """f_i(r) = (r / r_i) prod_{j != i} (r - r_j)/(r_i - r_j) / sqrt(a lam_i): the polynomial of degree nb that vanishes
    at r = 0, satisfies the Lagrange property f_i(r_j) = delta_ij / sqrt(lambda_j) (lambda_j = a lam_j on
    (0,a)).  Coefficients in mpmath from mpmath's OWN Gauss-Legendre nodes (not the oracle's)."""
    mp.mp.dps = dps
    nodes = sorted(mp.polyroots([mp.mpf(c) for c in mp.taylor(lambda t: mp.legendre(nb, t), 0, nb)[::-1]],
                                maxsteps=500, extraprec=400))
    xs = [(1 + t) / 2 for t in nodes]
    rs = [mp.mpf(a) * xx for xx in xs]
    lams = []
    for t in nodes:
        dp = mp.diff(lambda s: mp.legendre(nb, s), t)
        lams.append(1 / ((1 - t * t) * dp * dp))          # weight on (0,1): (2/((1-t^2)P'^2))/2
    polys = []
    for i in range(nb):
        c = [mp.mpf(1)]                                   # ascending coefficients
        for j in range(nb):
            if j == i:
                continue
            c = [(c[k - 1] if k >= 1 else 0) - rs[j] * (c[k] if k < len(c) else 0) for k in range(len(c) + 1)]
            den = rs[i] - rs[j]
            c = [v / den for v in c]
        c = [mp.mpf(0)] + c                               # multiply by r
        scale = 1 / (rs[i] * mp.sqrt(mp.mpf(a) * lams[i]))
        polys.append([v * scale for v in c])
    return xs, lams, polys


def _polyval(c, r):
    return sum(v * r ** k for k, v in enumerate(c))


def _polyder(c):
    return [k * v for k, v in enumerate(c)][1:]


def _polyint(c, lo, hi):
    return sum(v * (hi ** (k + 1) - lo ** (k + 1)) / (k + 1) for k, v in enumerate(c))


def _polymul(p, q):
    out = [mp.mpf(0)] * (len(p) + len(q) - 1)
    for i, a_ in enumerate(p):
        for j, b_ in enumerate(q):
            out[i + j] += a_ * b_
    return out


@pytest.mark.parametrize("nb,a", [(2, 1.0), (4, 10.0), (7, 3.5), (8, 20.0)])
def test_surface_values_and_kinetic_bloch_table_from_lagrange_polynomials(nb, a):
    xs, lams, polys = _lagrange_functions(nb, a)
    x, lam, r, fa = oracle.mesh(nb, a)
    T = oracle.kinetic(nb, a, x)
    assert np.allclose(x, [float(v) for v in xs], atol=4e-16)
    # q2(r_i) = f_i(a)
    fa_ref = np.array([float(_polyval(p, mp.mpf(a))) for p in polys])
    assert np.allclose(fa, fa_ref, rtol=1e-13)
    # <f_i| -d2/dr2 + delta(r-a) d/dr |f_j> = int_0^a f_i' f_j' dr   (f_i(0) = 0), exact polynomial integral
    Tref = np.zeros((nb, nb))
    for i in range(nb):
        for j in range(nb):
            Tref[i, j] = float(_polyint(_polymul(_polyder(polys[i]), _polyder(polys[j])), mp.mpf(0), mp.mpf(a)))
    assert np.allclose(T, Tref, rtol=1e-12, atol=1e-12 * np.abs(Tref).max())
    assert np.array_equal(T, T.T)
    # the same matrix element written the other way: -int f_i f_j'' + f_i(a) f_j'(a)
    i, j = 0, nb - 1
    d2 = _polyder(_polyder(polys[j]))
    alt = -_polyint(_polymul(polys[i], d2), mp.mpf(0), mp.mpf(a)) + _polyval(polys[i], mp.mpf(a)) * _polyval(
        _polyder(polys[j]), mp.mpf(a))
    assert abs(float(alt) - T[i, j]) < 1e-12 * np.abs(Tref).max()


def test_lagrange_property_of_reference_polynomials():
    """Sanity of the test's own reference: f_i(r_j) = delta_ij / sqrt(a lam_j), orthonormal at Gauss accuracy."""
    nb, a = 5, 2.0
    xs, lams, polys = _lagrange_functions(nb, a)
    for i in range(nb):
        for j in range(nb):
            v = _polyval(polys[i], a * xs[j])
            ref = (1 / mp.sqrt(a * lams[j])) if i == j else 0
            assert abs(v - ref) < mp.mpf(10) ** -30


# ----------------------------------------------------------------- assembly structure (PAPER.md:87-99 Eqs. 3,4; :137)

def _small_system(nch=3, nb=4, seed=5, symmetric=False):
    rng = np.random.default_rng(seed)
    a, h2m = 6.0, 11.0
    lval = np.array([2, 0, 1][:nch], dtype=np.int32)
    ethr = np.array([0.0, 0.7, 1.9][:nch])
    V = rng.normal(size=(nb, nch, nch)) + 1j * rng.normal(size=(nb, nch, nch))
    if symmetric:
        V = (V + V.transpose(0, 2, 1)) / 2
    return a, h2m, lval, ethr, V


def test_assemble_block_structure_and_index_convention():
    nch, nb, E = 3, 4, 2.5
    a, h2m, lval, ethr, V = _small_system(nch, nb)
    C = oracle.assemble(nch, nb, a, h2m, lval, ethr, E, V)
    x, lam, r, fa = oracle.mesh(nb, a)
    T = oracle.kinetic(nb, a, x)
    for c1, c2 in itertools.product(range(nch), repeat=2):
        blk = C[c1 * nb:(c1 + 1) * nb, c2 * nb:(c2 + 1) * nb]       # row = i + c*nb (PAPER.md:137 step 4)
        if c1 != c2:
            # Eq. (4): D_cc' diagonal with V_cc'(r_i); V[i, c2, c1] = V_{c1 c2}(r_i)
            assert np.array_equal(blk, np.diag(V[:, c2, c1]))
        else:
            off = blk - np.diag(np.diag(blk))
            assert np.array_equal(off, h2m * (T - np.diag(np.diag(T))))
            want = h2m * np.diag(T) + h2m * lval[c1] * (lval[c1] + 1) / r ** 2 + (ethr[c1] - E) + V[:, c1, c1]
            assert np.allclose(np.diag(blk), want, rtol=1e-15)
    # energy enters as -E on the whole diagonal and nowhere else (C - E I)
    C0 = oracle.assemble(nch, nb, a, h2m, lval, ethr, 0.0, V)
    assert np.allclose(C0 - C, E * np.eye(nch * nb), atol=1e-12)


def test_rhs_layout():
    nch, nb = 3, 4
    _, _, _, fa = oracle.mesh(nb, 6.0)
    B = oracle.rhs(nch, nb, fa)
    for c in range(nch):
        col = np.zeros(nch * nb)
        col[c * nb:(c + 1) * nb] = fa
        assert np.array_equal(B[:, c], col)


# ----------------------------------------------------------------- LU / solve (Eq. 5)

def _cramer(A, b):
    mp.mp.dps = 40
    n = A.shape[0]
    Am = mp.matrix(n, n)
    for i in range(n):
        for j in range(n):
            Am[i, j] = mp.mpc(A[i, j])

    def det(M):  # cofactor expansion, written out (no LU inside)
        m = M.rows
        if m == 1:
            return M[0, 0]
        s = mp.mpc(0)
        for j in range(m):
            minor = mp.matrix(m - 1, m - 1)
            for ii in range(1, m):
                cc = 0
                for jj in range(m):
                    if jj == j:
                        continue
                    minor[ii - 1, cc] = M[ii, jj]
                    cc += 1
            s += (-1) ** j * M[0, j] * det(minor)
        return s

    d = det(Am)
    x = []
    for k in range(n):
        Ak = Am.copy()
        for i in range(n):
            Ak[i, k] = mp.mpc(b[i])
        x.append(complex(det(Ak) / d))
    return np.array(x)


def _gauss_jordan_inverse(A):
    mp.mp.dps = 40
    n = A.shape[0]
    M = [[mp.mpc(A[i, j]) for j in range(n)] + [mp.mpc(1 if i == j else 0) for j in range(n)] for i in range(n)]
    for c in range(n):
        p = max(range(c, n), key=lambda rr: abs(M[rr][c]))
        M[c], M[p] = M[p], M[c]
        pv = M[c][c]
        M[c] = [v / pv for v in M[c]]
        for rr in range(n):
            if rr != c:
                f = M[rr][c]
                M[rr] = [v - f * w for v, w in zip(M[rr], M[c])]
    return np.array([[complex(M[i][n + j]) for j in range(n)] for i in range(n)])


@pytest.mark.parametrize("n,seed", [(1, 0), (2, 1), (3, 2), (5, 3), (7, 4)])
@pytest.mark.parametrize("mode,nrefine", [(0, 0), (1, 0), (0, 2)])
def test_solve_against_cramers_rule(n, seed, mode, nrefine):
    rng = np.random.default_rng(seed)
    A = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    A[0, 0] = 0.0                                            # forces a row interchange at step 0 when n > 1
    if n == 1:
        A[0, 0] = 0.3 - 2j
    B = rng.normal(size=(n, 2)) + 1j * rng.normal(size=(n, 2))
    X = oracle.solve(A, B, mode=mode, nrefine=nrefine)
    for q in range(2):
        assert np.allclose(X[:, q], _cramer(A, B[:, q]), rtol=1e-12, atol=1e-13)


@pytest.mark.parametrize("n", [4, 8])
def test_solve_against_explicit_gauss_jordan_inverse(n):
    rng = np.random.default_rng(100 + n)
    A = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    B = rng.normal(size=(n, 3)) + 1j * rng.normal(size=(n, 3))
    X = oracle.solve(A, B, nrefine=0)
    assert np.allclose(X, _gauss_jordan_inverse(A) @ B, rtol=1e-12, atol=1e-13)


def test_solve_pivots_are_valid_and_first_max():
    rng = np.random.default_rng(9)
    n = 40
    A = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    X, ipiv = oracle.solve(A, np.eye(n, dtype=complex), nrefine=0, return_ipiv=True)
    assert np.all(ipiv >= np.arange(n)) and np.all(ipiv < n)
    col0 = np.abs(A[:, 0].real) + np.abs(A[:, 0].imag)
    assert ipiv[0] == int(np.argmax(col0))
    assert np.allclose(A @ X, np.eye(n), atol=1e-11)


def test_solve_singular_matrix_is_reported():
    A = np.array([[1, 2], [2, 4]], dtype=complex)
    with pytest.raises(ZeroDivisionError):
        oracle.solve(A, np.ones((2, 1), dtype=complex))


@pytest.mark.parametrize("n", [64, 300])
def test_manufactured_solution_x_equals_one(n):
    """PAPER.md:563 (Table 7 caption): x_exact = 1, b = A 1."""
    rng = np.random.default_rng(n)
    A = rng.uniform(-1, 1, size=(n, n)) + 1j * rng.uniform(-1, 1, size=(n, n)) + np.sqrt(n) * np.eye(n)
    b = A @ np.ones((n, 1))
    for mode in (0, 1):
        X = oracle.solve(A, b, mode=mode, nrefine=2)
        assert np.abs(X - 1).max() < 1e-14


def test_structured_residual_equals_dense_residual():
    nch, nb, E = 3, 6, 1.3
    a, h2m, lval, ethr, V = _small_system(nch, nb, seed=11)
    C = oracle.assemble(nch, nb, a, h2m, lval, ethr, E, V)
    rng = np.random.default_rng(0)
    X = np.asfortranarray(rng.normal(size=(nch * nb, nch)) + 1j * rng.normal(size=(nch * nb, nch)))
    _, _, _, fa = oracle.mesh(nb, a)
    B = oracle.rhs(nch, nb, fa)
    r1 = oracle.structured_residual(nch, nb, a, h2m, lval, ethr, E, V, X)
    r2 = B - np.asarray(C, dtype=np.clongdouble) @ np.asarray(X, dtype=np.clongdouble)
    assert np.allclose(r1, r2.astype(complex), rtol=0, atol=1e-13 * np.abs(C).max())
    Bx = np.asfortranarray(rng.normal(size=X.shape) + 0j)
    r3 = oracle.structured_residual(nch, nb, a, h2m, lval, ethr, E, V, X, B=Bx)
    assert np.allclose(r3 - r1, Bx - B, atol=1e-12 * np.abs(C).max())


# ----------------------------------------------------------------- whole chain: closed forms

@pytest.mark.parametrize("l", [0, 1, 2, 3])
def test_free_particle_R_matrix_and_zero_phase_shift(l):
    """V = 0: R = F_l(ka)/(ka F_l'(ka)), S = 1, phase shift 0."""
    nb, a, E = 30, 10.0, 10.0
    k = np.sqrt(E / H2M)
    V = np.zeros((nb, 1, 1), dtype=complex)
    R = oracle.rmatrix(1, nb, a, H2M, [l], [0.0], E, V)
    want = R_constant_potential(l, k, a)
    assert abs(R[0, 0] - want) < 1e-11 * abs(want)
    S = smatrix(R, [l], np.array([k]), a)
    assert abs(S[0, 0] - 1.0) < 1e-10
    assert abs(0.5 * np.angle(S[0, 0])) < 1e-10


def test_square_well_phase_shift_converges_with_nb():
    """Constant well of depth V0 filling (0,a), l = 0: R = tan(Ka)/(Ka), tan(ka + delta) = (k/K) tan(Ka).
    Error falls exponentially with nb (Gauss quadrature is exact for the polynomial basis)."""
    a, E, V0 = 10.0, 10.0, 50.0
    k, K = np.sqrt(E / H2M), np.sqrt((E + V0) / H2M)
    Rex = np.tan(K * a) / (K * a)
    delta_ex = np.arctan((k / K) * np.tan(K * a)) - k * a
    errs = []
    for nb in (10, 15, 20, 25):
        V = np.full((nb, 1, 1), -V0, dtype=complex)
        R = oracle.rmatrix(1, nb, a, H2M, [0], [0.0], E, V)
        errs.append(abs(R[0, 0] - Rex) / abs(Rex))
        S = smatrix(R, [0], np.array([k]), a)
        d = 0.5 * np.angle(S[0, 0])
        derr = abs(np.exp(2j * d) - np.exp(2j * delta_ex))
        if nb >= 20:
            assert derr < 1e-9
    assert errs[0] > 1e-3 and errs[1] < errs[0] * 1e-2 and errs[2] < 1e-9 and errs[3] < 1e-10


def test_uncoupled_channels_with_thresholds_and_complex_well():
    """Diagonal V: every channel is an independent constant-potential problem with its own l_c and E - E_c (the
    threshold enters as +E_c on the diagonal); absorptive (complex) wells and a CLOSED channel included."""
    nb, a, E = 40, 8.0, 6.0
    lval = [0, 2, 1, 3]
    ethr = [0.0, 1.5, 3.0, 9.0]                                 # last channel closed (E < E_c)
    depth = [30.0 + 5j, 12.0, 0.0, 20.0 + 1j]
    V = np.zeros((nb, 4, 4), dtype=complex)
    for c in range(4):
        V[:, c, c] = -depth[c]
    R = oracle.rmatrix(4, nb, a, H2M, lval, ethr, E, V)
    assert np.abs(R - np.diag(np.diag(R))).max() == 0.0
    for c in range(4):
        K = np.sqrt(complex((E - ethr[c] + depth[c]) / H2M))
        want = R_constant_potential(lval[c], K, a)
        assert abs(R[c, c] - want) < 2e-10 * abs(want), c


def test_constant_nonsymmetric_coupling_matrix_pins_channel_index_order():
    """All channels share l and threshold, V(r) = W constant and NON-symmetric, W = P diag(w) P^-1.  Then the system
    decouples in the eigenbasis: R = P diag(R_l(K_m)) P^-1 with K_m = sqrt((E - w_m)/h2m).  A transposed V index
    (c1 <-> c2) would give R^T instead."""
    nb, a, E, l = 40, 8.0, 6.0, 1
    rng = np.random.default_rng(3)
    P = rng.normal(size=(3, 3)) + 2 * np.eye(3)
    w = np.array([-20.0 - 3j, -5.0, 1.0 - 0.5j])
    W = P @ np.diag(w) @ np.linalg.inv(P)
    V = np.empty((nb, 3, 3), dtype=complex)
    V[:] = W.T[None]                                             # V[i, c2, c1] = W[c1, c2]
    R = oracle.rmatrix(3, nb, a, H2M, [l] * 3, [0.0] * 3, E, V)
    Rm = np.array([R_constant_potential(l, np.sqrt(complex((E - wm) / H2M)), a) for wm in w])
    want = P @ np.diag(Rm) @ np.linalg.inv(P)
    assert np.abs(R - want).max() < 1e-9 * np.abs(want).max()
    assert np.abs(R - want.T).max() > 1e-3 * np.abs(want).max()


# ----------------------------------------------------------------- whole chain: invariants at config 0

def test_cfg0_R_symmetric_and_S_subunitary_and_big_n_mode_agrees():
    w = make_workload(0)
    x, lam, r, fa = oracle.mesh(w.nb, w.a)
    V = w.potential(r)
    E = float(w.energies[0])
    R = oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, V)
    assert np.abs(R - R.T).max() < 1e-13 * np.abs(R).max()       # C = C^T  =>  R = R^T
    k = np.sqrt((E - w.ethr) / w.h2m)
    S = smatrix(R, w.lval, k, w.a)
    assert np.abs(S - S.T).max() < 1e-11
    sv = np.linalg.svd(S, compute_uv=False)
    assert sv.max() < 1.0                                        # W0 > 0: absorption
    R1 = oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, V, mode=1)
    assert np.abs(R1 - R).max() < 1e-13 * np.abs(R).max()        # big-N mode validation


def test_cfg0_real_potential_gives_unitary_S():
    w = make_workload(0)
    w.W0 = 0.0
    x, lam, r, fa = oracle.mesh(w.nb, w.a)
    V = w.potential(r)
    E = float(w.energies[0])
    R = oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, V)
    assert np.abs(R.imag).max() < 1e-13 * np.abs(R).max()
    S = smatrix(R, w.lval, np.sqrt((E - w.ethr) / w.h2m), w.a)
    assert np.abs(S.conj().T @ S - np.eye(w.nch)).max() < 1e-11


def test_rmatrix_equals_definition_via_dense_solve_and_certificate():
    """R = (h2m/a) B^T (C - E)^-1 B computed the long way (assemble -> dense solve -> contract) equals orc_rmatrix, and
    the a-posteriori certificate (h2m/a) X^T (B - C X) of SURVEY 8(c) is ~0 for the oracle's own X."""
    w = make_workload(0, nch=3, nb=20)
    x, lam, r, fa = oracle.mesh(w.nb, w.a)
    V = w.potential(r)
    E = 7.0
    R, X = oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, V, return_x=True)
    C = oracle.assemble(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, V)
    B = oracle.rhs(w.nch, w.nb, fa)
    X2 = oracle.solve(C, B, nrefine=2)
    R2 = oracle.contract(w.nch, w.nb, w.a, w.h2m, fa, X2)
    assert np.abs(R2 - R).max() < 1e-14 * np.abs(R).max()
    assert np.allclose(R2, (w.h2m / w.a) * B.T @ X2, rtol=1e-13, atol=1e-16)
    res = oracle.structured_residual(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, V, X)
    cert = (w.h2m / w.a) * X.T @ res
    assert np.abs(cert).max() < 1e-13 * np.abs(R).max()


# ----------------------------------------------------------------- collision matrix (neutral case)
def _ws_potential(nb, a, nch, beta, V0=50.0, W0=0.0, Rws=3.0, aws=0.65):
    r = oracle.mesh(nb, a)[2]
    u = np.exp((r - Rws) / aws)
    f, df = 1.0 / (1.0 + u), -u / (aws * (1.0 + u) ** 2)
    V = np.zeros((nb, nch, nch), dtype=complex)
    for i in range(nb):
        V[i] = beta * df[i]
        V[i][np.diag_indices(nch)] = -(V0 + 1j * W0) * f[i]
    return V


def test_collision_matrix_free_particles_scatter_nothing_closed_channel_present():
    """V = 0 with thresholds, one channel closed: U = 1 on the open channels (pins signs, derivatives and the k^-1/2
    normalisation of the matching formula)."""
    nb, a, E = 40, 8.0, 6.0
    lval, ethr = [0, 2, 1, 3], [0.0, 1.5, 3.0, 9.0]
    R = oracle.rmatrix(4, nb, a, H2M, lval, ethr, E, np.zeros((nb, 4, 4), dtype=complex))
    U, opn = oracle.collision_matrix(R, lval, ethr, E, H2M, a)
    assert list(opn) == [0, 1, 2]
    assert np.abs(U - np.eye(3)).max() < 1e-9


def test_collision_matrix_unitary_and_symmetric_with_a_closed_channel():
    """Real symmetric couplings, one closed channel: flux conservation among the OPEN channels (U^dagger U = 1) holds only if
    the closed channel is matched to the decaying function; U = U^T from C = C^T.  With absorption (W0 > 0) all singular
    values drop below 1."""
    nb, a, E = 40, 8.0, 6.0
    lval, ethr = [0, 2, 1, 3], [0.0, 1.5, 3.0, 9.0]
    rng = np.random.default_rng(3)
    beta = rng.uniform(5.0, 20.0, (4, 4))
    beta = 0.5 * (beta + beta.T)
    np.fill_diagonal(beta, 0.0)
    R = oracle.rmatrix(4, nb, a, H2M, lval, ethr, E, _ws_potential(nb, a, 4, beta))
    U, opn = oracle.collision_matrix(R, lval, ethr, E, H2M, a)
    assert len(opn) == 3 and np.abs(U).max() < 1.0 + 1e-12 and np.abs(U[0, 1]) > 0.05      # genuinely coupled
    assert np.abs(U.conj().T @ U - np.eye(3)).max() < 1e-12
    assert np.abs(U - U.T).max() < 1e-12
    Ra = oracle.rmatrix(4, nb, a, H2M, lval, ethr, E, _ws_potential(nb, a, 4, beta, W0=10.0))
    Ua, _ = oracle.collision_matrix(Ra, lval, ethr, E, H2M, a)
    assert np.linalg.svd(Ua, compute_uv=False).max() < 1.0 - 1e-3


def test_collision_matrix_reduces_to_the_all_open_formula_and_ignores_a_decoupled_closed_channel():
    nb, a = 40, 8.0
    lval, ethr = [0, 2, 1, 3], [0.0, 1.5, 3.0, 9.0]
    rng = np.random.default_rng(4)
    beta = rng.uniform(5.0, 20.0, (4, 4))
    beta = 0.5 * (beta + beta.T)
    np.fill_diagonal(beta, 0.0)
    V = _ws_potential(nb, a, 4, beta)
    # all channels open: the independent test-side helper (scatter.smatrix) gives the same matrix
    E = 12.0
    R = oracle.rmatrix(4, nb, a, H2M, lval, ethr, E, V)
    U, opn = oracle.collision_matrix(R, lval, ethr, E, H2M, a)
    assert len(opn) == 4
    assert np.abs(U - smatrix(R, lval, np.sqrt((E - np.array(ethr)) / H2M), a)).max() < 1e-12
    # a closed channel that is not coupled to the others cannot change their collision matrix
    E = 6.0
    V3 = V.copy()
    V3[:, 3, :3] = 0.0
    V3[:, :3, 3] = 0.0
    R4 = oracle.rmatrix(4, nb, a, H2M, lval, ethr, E, V3)
    R3 = oracle.rmatrix(3, nb, a, H2M, lval[:3], ethr[:3], E, np.ascontiguousarray(V3[:, :3, :3]))
    U4, _ = oracle.collision_matrix(R4, lval, ethr, E, H2M, a)
    U3, _ = oracle.collision_matrix(R3, lval[:3], ethr[:3], E, H2M, a)
    assert np.abs(U4 - U3).max() < 1e-12


def test_collision_matrix_stays_unitary_far_below_the_centrifugal_barrier():
    """l = 12 at k a = 0.56 (G/F ~ 1e27): flux conservation and symmetry to rounding, which the literal (Z^O)^-1 Z^I form
    cannot deliver in FP64 (reading R14); the barely penetrable channel decouples, |U_11| = 1."""
    nb, a, E = 40, 8.0, 6.0
    lval, ethr = [0, 12, 1], [0.0, 5.9, 3.0]
    beta = np.array([[0.0, 12.0, 9.0], [12.0, 0.0, 15.0], [9.0, 15.0, 0.0]])
    R = oracle.rmatrix(3, nb, a, H2M, lval, ethr, E, _ws_potential(nb, a, 3, beta))
    U, opn = oracle.collision_matrix(R, lval, ethr, E, H2M, a)
    assert len(opn) == 3
    assert np.abs(U.conj().T @ U - np.eye(3)).max() < 1e-12
    assert np.abs(U - U.T).max() < 1e-12
    assert abs(abs(U[1, 1]) - 1.0) < 1e-12 and np.abs(U[1, [0, 2]]).max() < 1e-15
    assert np.abs(U[0, 2]) > 1e-3


def test_collision_matrix_equals_the_literal_definition_in_60_digit_arithmetic():
    """The oracle evaluates U = 1 - 2i (Z^O)^-1 Z^F; reading R14's DEFINITION is U = (Z^O)^-1 Z^I with
    Z^O_cc' = (k_c' a)^-1/2 [O_c delta_cc' - R_cc' x_c' O'_c'(x_c')] and Z^I likewise with I = G - iF.  Here the literal
    definition is evaluated in mpmath at 60 digits (Riccati-Bessel functions from mpmath's besselj / bessely, derivatives by
    the recurrence f_l' = f_{l-1} - (l/x) f_l, an mpmath LU solve) on the sub-barrier case l = 12, k a = 0.56 -- where the
    literal form loses everything in FP64 -- and on an ordinary case; the oracle must agree to 1e-12."""
    import mpmath as mp

    def literal(R, lval, ethr, E, a):
        with mp.workdps(60):
            n = len(lval)
            x = [mp.sqrt((mp.mpf(E) - mp.mpf(float(e))) / mp.mpf(H2M)) * mp.mpf(a) for e in ethr]   # all channels open here
            half = mp.mpf(1) / 2
            Ff = lambda l, t: mp.sqrt(mp.pi * t / 2) * mp.besselj(l + half, t)       # F_l(t) = t j_l(t)
            Gf = lambda l, t: -mp.sqrt(mp.pi * t / 2) * mp.bessely(l + half, t)      # G_l(t) = -t y_l(t)
            O, dO, I, dI = [], [], [], []
            for l, t in zip(lval, x):
                F, G = Ff(l, t), Gf(l, t)
                # Riccati-Bessel recurrence u_l' = u_{l-1} - (l/t) u_l  
                dF = Ff(l - 1, t) - l / t * F
                dG = Gf(l - 1, t) - l / t * G
                O.append(G + 1j * F)
                dO.append(t * (dG + 1j * dF))
                I.append(G - 1j * F)
                dI.append(t * (dG - 1j * dF))
            Rm = mp.matrix(n, n)
            for i in range(n):
                for j in range(n):
                    Rm[i, j] = mp.mpc(complex(R[i, j]))
            ZO, ZI = mp.matrix(n, n), mp.matrix(n, n)
            for i in range(n):
                for j in range(n):
                    s = 1 / mp.sqrt(x[j])
                    ZO[i, j] = ((O[i] if i == j else 0) - Rm[i, j] * dO[j]) * s
                    ZI[i, j] = ((I[i] if i == j else 0) - Rm[i, j] * dI[j]) * s
            cols = [mp.lu_solve(ZO, ZI[:, j]) for j in range(n)]
            return np.array([[complex(cols[j][i]) for j in range(n)] for i in range(n)])

    nb, a = 40, 8.0
    cases = [([0, 12, 1], [0.0, 5.9, 3.0], 6.0,                                       # k a = 0.56 in the l = 12 channel
              np.array([[0.0, 12.0, 9.0], [12.0, 0.0, 15.0], [9.0, 15.0, 0.0]])),
             ([0, 2, 1], [0.0, 1.5, 3.0], 12.0,
              np.array([[0.0, 7.0, 11.0], [7.0, 0.0, 5.0], [11.0, 5.0, 0.0]]))]
    for lval, ethr, E, beta in cases:
        R = oracle.rmatrix(3, nb, a, H2M, lval, ethr, E, _ws_potential(nb, a, 3, beta))
        U, opn = oracle.collision_matrix(R, lval, ethr, E, H2M, a)
        assert len(opn) == 3
        assert np.abs(U - literal(R, lval, ethr, E, a)).max() < 1e-12, (lval, E)


# ----------------------------------------------------------------- charged case: Coulomb / Whittaker functions
E2 = 1.43996  # e^2, MeV fm


def test_coulomb_channel_functions_wronskian_and_neutral_limit():
    """F'G - FG' = 1 (A&S 14.2.4) for the pair the oracle builds (function values and recurrence derivatives come from
    different mpmath evaluations), and eta = 0 reproduces the Riccati-Bessel functions of the neutral branch."""
    from oracle.oracle import _coulomb_channel
    from scipy.special import spherical_jn, spherical_yn, spherical_kn
    for l, eta, x in itertools.product([0, 1, 4, 11], [0.0, 0.3, 2.5, 8.0], [0.7, 4.0, 25.0]):
        F, xdF, G, xdG = _coulomb_channel(l, eta, x, True)
        assert abs((xdF * G - F * xdG) / x - 1.0) < 1e-12
    for l, x in itertools.product([0, 2, 7], [0.5, 3.0, 12.0]):
        F, xdF, G, xdG = _coulomb_channel(l, 0.0, x, True)
        assert abs(F - x * spherical_jn(l, x)) < 1e-13 * max(1, abs(F)) and abs(G + x * spherical_yn(l, x)) < 1e-13 * abs(G)
        _, _, one, xdW = _coulomb_channel(l, 0.0, x, False)
        k, dk = spherical_kn(l, x), spherical_kn(l, x, derivative=True)
        assert one == 1.0 and abs(xdW - x * (k + x * dk) / (x * k)) < 1e-12 * abs(xdW)


def test_collision_matrix_charged_branch_reduces_to_neutral():
    rng = np.random.default_rng(0)
    R = rng.normal(size=(4, 4)) * 0.1
    R = R + R.T + 0j
    lval, ethr = [0, 2, 1, 3], [0.0, 1.5, 3.0, 9.0]
    U0, _ = oracle.collision_matrix(R, lval, ethr, 6.0, H2M, 8.0)
    U1, _ = oracle.collision_matrix(R, lval, ethr, 6.0, H2M, 8.0, zze2=[1e-300] * 4)     # forces the mpmath branch
    assert np.abs(U0 - U1).max() < 1e-13


def test_pure_coulomb_potential_scatters_nothing_relative_to_coulomb_waves():
    """V_cc(r) = Z1 Z2 e^2 / r and nothing else, a different charge product per channel: the internal solution IS the
    regular Coulomb function, so U = 1 (pins eta = zze2 / (2 h2m k), the Coulomb functions, their derivatives and the
    per-channel indexing; accuracy = convergence of the Nb = 60 mesh)."""
    nb, a, E = 60, 8.0, 6.0
    lval, ethr = [0, 2, 1, 3], [0.0, 1.5, 3.0, 9.0]
    zz = [2 * E2, 4 * E2, 1 * E2, 6 * E2]
    r = oracle.mesh(nb, a)[2]
    V = np.zeros((nb, 4, 4), dtype=complex)
    for c in range(4):
        V[:, c, c] = zz[c] / r
    R = oracle.rmatrix(4, nb, a, H2M, lval, ethr, E, V)
    U, opn = oracle.collision_matrix(R, lval, ethr, E, H2M, a, zze2=zz)
    assert list(opn) == [0, 1, 2]
    assert np.abs(U - np.eye(3)).max() < 1e-8


@pytest.mark.parametrize("zz", [0.0, 3 * E2])
def test_collision_matrix_does_not_depend_on_the_channel_radius(zz):
    """Beyond the range of the nuclear potential U is independent of a -- but only if every channel is matched to the
    right external solution: this pins the CLOSED-channel function (x k_l(x) / Whittaker), whose logarithmic derivative no
    unitarity or decoupling test can see.  The closed channel lies 0.3 MeV below the energy (kappa a ~ 1), so its tail at a
    is large: the correct functions agree to 1e-9 between the two radii, the growing solution gives 6e-4, eta dropped 5e-6,
    a logarithmic derivative 5 % off 2e-6 (checked when the pin was written)."""
    lval, ethr, E = [0, 1, 2], [0.0, 2.0, 6.3], 6.0
    beta = np.array([[0.0, 30.0, 40.0], [30.0, 0.0, 35.0], [40.0, 35.0, 0.0]])
    Us = []
    for a, nb in [(9.0, 90), (11.0, 110)]:
        r = oracle.mesh(nb, a)[2]
        V = _ws_potential(nb, a, 3, beta, Rws=2.5, aws=0.25)
        for c in range(3):
            V[:, c, c] += zz / r
        R = oracle.rmatrix(3, nb, a, H2M, lval, ethr, E, V)
        U, opn = oracle.collision_matrix(R, lval, ethr, E, H2M, a, zze2=[zz] * 3 if zz else None)
        assert list(opn) == [0, 1]
        assert np.abs(U.conj().T @ U - np.eye(2)).max() < 1e-10
        Us.append(U)
    assert np.abs(Us[0][0, 1]) > 0.05
    assert np.abs(Us[0] - Us[1]).max() < 5e-8


# ----------------------------------------------------------------- non-local potentials
def test_nonlocal_with_a_local_kernel_is_the_local_path():
    """W = V(r_i) delta_ij in every block must reproduce rmatrix() (pins the index convention of W and the diagonal part)."""
    w = make_workload(0, nch=3, nb=30)
    E = 7.0
    r = oracle.mesh(w.nb, w.a)[2]
    V = w.potential(r)
    W = np.zeros((w.n, w.n), dtype=complex)
    for c1, c2 in itertools.product(range(3), range(3)):
        W[c1 * w.nb + np.arange(w.nb), c2 * w.nb + np.arange(w.nb)] = V[:, c2, c1]
    Rn = oracle.rmatrix_nonlocal(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, W)
    Rl = oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, V)
    assert np.abs(Rn - Rl).max() < 1e-13 * np.abs(Rl).max()


@pytest.mark.parametrize("E", [0.5, 5.0, 30.0])
def test_separable_potential_has_the_analytic_phase_shift(E):
    """Rank-one kernel W(r,r') = -lambda exp(-beta r) exp(-beta r') (the s-wave Yamaguchi form), acting on u = r psi:
    u'' + k^2 u = -Lambda c exp(-beta r), c = int_0^inf exp(-beta r) u dr, Lambda = lambda/h2m, solved by hand:
        tan(delta) = Lambda k / [ (beta^2 + k^2)^2 + Lambda (k^2 - beta^2) / (2 beta) ].
    A genuinely non-local problem with a closed form: pins the Gauss approximation a sqrt(lam_i lam_j) W(r_i, r_j), the full
    (not diagonal) use of W, and the sign of the potential."""
    nb, a, beta, lam0 = 60, 12.0, 2.0, 400.0
    x, lam, r, fa = oracle.mesh(nb, a)
    W = -lam0 * a * np.sqrt(np.outer(lam, lam)) * np.exp(-beta * (r[:, None] + r[None, :])) + 0j
    R = oracle.rmatrix_nonlocal(1, nb, a, H2M, [0], [0.0], E, W)
    U, _ = oracle.collision_matrix(R, [0], [0.0], E, H2M, a)
    k = np.sqrt(E / H2M)
    Lam = lam0 / H2M
    tan_d = Lam * k / ((beta ** 2 + k ** 2) ** 2 + Lam * (k ** 2 - beta ** 2) / (2 * beta))
    S_exact = (1 + 1j * tan_d) / (1 - 1j * tan_d)
    assert abs(abs(U[0, 0]) - 1.0) < 1e-12
    assert abs(tan_d) > 0.05
    assert abs(U[0, 0] - S_exact) < 1e-8


# ----------------------------------------------------------------- propagation over sub-intervals (reading R16)
def test_sector_matrices_of_free_motion_match_the_closed_form():
    """V = 0, l = 0 on (a_lo, a_hi), h = a_hi - a_lo: u = A cos k(r - a_lo) + B sin k(r - a_lo) gives
    u(a_hi) = -cot(kh)/k u'(a_hi) + 1/(k sin kh) u'(a_lo),  u(a_lo) = -1/(k sin kh) u'(a_hi) + cot(kh)/k u'(a_lo), i.e.
    Rsec_RR = Rsec_LL = -cot(kh)/k, Rsec_RL = Rsec_LR = -1/(k sin kh).  Pins the sector mesh, the two-sided Bloch kinetic
    matrix, both surface vectors and the sign convention of the four blocks."""
    a_lo, a_hi, E, nb = 3.0, 7.5, 11.0, 30
    k = np.sqrt(E / H2M)
    h = a_hi - a_lo
    (LL, LR), (RL, RR) = oracle.sector_matrices(1, nb, a_lo, a_hi, H2M, [0], [0.0], E, np.zeros((nb, 1, 1), dtype=complex))
    d, o = -1 / (k * np.tan(k * h)), -1 / (k * np.sin(k * h))
    assert abs(RR[0, 0] - d) < 1e-11 * abs(d) and abs(LL[0, 0] - d) < 1e-11 * abs(d)
    assert abs(RL[0, 0] - o) < 1e-11 * abs(o) and abs(LR[0, 0] - o) < 1e-11 * abs(o)


def test_sector_tables_lagrange_and_symmetry_properties():
    nb, a_lo, a_hi = 12, 2.0, 5.0
    r, faL, faR, T = oracle.sector_tables(nb, a_lo, a_hi)
    x, lam, _, _ = oracle.mesh(nb, 1.0)
    assert np.allclose(r, a_lo + (a_hi - a_lo) * x, rtol=1e-15)
    assert np.allclose(T, T.T, rtol=0, atol=1e-12 * np.abs(T).max())
    # sum_i sqrt(h lam_i) f_i(r) = 1 (the Lagrange polynomials sum to one): at both ends, and its derivative vanishes: T 1~ = 0
    w = np.sqrt((a_hi - a_lo) * lam)
    assert abs(np.dot(w, faL) - 1) < 1e-12 and abs(np.dot(w, faR) - 1) < 1e-12
    assert np.abs(T @ w).max() < 1e-10 * np.abs(T).max()


@pytest.mark.parametrize("lval,Vdepth", [([0], 0.0), ([2], 0.0), ([3], 30.0)])
def test_propagated_rmatrix_matches_the_closed_form_of_a_constant_potential(lval, Vdepth):
    """R at a_2 obtained from the single-interval R at a_1 and the sector (a_1, a_2) must be F_l(K a_2)/(K a_2 F_l'(K a_2)):
    sees the centrifugal term on the shifted mesh and the propagation formula."""
    a1, a2, E, nb = 4.0, 9.0, 13.0, 40
    V1 = np.full((nb, 1, 1), -Vdepth, dtype=complex)
    R1 = oracle.rmatrix(1, nb, a1, H2M, lval, [0.0], E, V1)
    Rsec = oracle.sector_matrices(1, nb, a1, a2, H2M, lval, [0.0], E, V1)
    R2 = oracle.propagate(a1, a2, R1, Rsec)
    K = np.sqrt((E + Vdepth) / H2M)
    assert abs(R2[0, 0] - R_constant_potential(lval[0], K, a2)) < 1e-9 * max(1.0, abs(R2[0, 0]))


def test_propagation_over_two_sub_intervals_equals_the_single_interval_rmatrix():
    """Coupled channels with a closed one and absorption: R(a) from (0, a/2) + (a/2, a) equals R(a) from (0, a) up to the
    discretisation error of the two meshes (both converged here), and stays symmetric."""
    w = make_workload(0)
    a1, E, nb = 0.45 * w.a, 2.5, 50
    r_full = oracle.mesh(nb, w.a)[2]
    R_full = oracle.rmatrix(w.nch, nb, w.a, w.h2m, w.lval, w.ethr, E, make_workload(0, nb=nb).potential(r_full))
    wl = make_workload(0, nb=nb)
    R1 = oracle.rmatrix(w.nch, nb, a1, w.h2m, w.lval, w.ethr, E, wl.potential(oracle.mesh(nb, a1)[2]))
    rs = oracle.sector_tables(nb, a1, w.a)[0]
    Rsec = oracle.sector_matrices(w.nch, nb, a1, w.a, w.h2m, w.lval, w.ethr, E, wl.potential(rs))
    R2 = oracle.propagate(a1, w.a, R1, Rsec)
    assert np.abs(R2 - R_full).max() / np.abs(R_full).max() < 1e-8
    assert np.abs(R2 - R2.T).max() < 1e-11 * np.abs(R2).max()
    assert np.abs(Rsec[0][1] - Rsec[1][0].T).max() < 1e-11 * np.abs(Rsec[0][1]).max()
