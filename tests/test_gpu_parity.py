"""Parity of the CUDA path (through the C ABI, include/hprmat.h) with the CPU oracle, element by element on the same
seeded inputs.  All tests here need a B200 ("-m gpu").

Tolerances (BASELINE.json north_star; norms per DESIGN.md readings R7/R8):
  FP64 path: max|R - R_orc| / max|R_orc| <= 1e-10, backward error <= 50 N 2^-53;
  assembly: every entry within 4 ulp of the oracle's (the two sides evaluate the closed forms independently in long
  double and round once; the FP64 evaluation order of the diagonal is fixed by reading R4), structural zeros exact;
  integer/index work (pivots): validity of P A = L U, since ties make the pivot sequence non-unique (reading R6).
"""
import numpy as np
import pytest
import torch

import oracle
from certificate import certificate
from paper_2512_11590_b200 import binding as hb
from paper_2512_11590_b200.workloads import dense_test_matrix, make_workload

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _dev_colmajor(a: np.ndarray) -> torch.Tensor:
    """numpy (m, n) -> torch CUDA tensor of shape (n, m) whose memory is the column-major m x n matrix."""
    return torch.from_numpy(np.ascontiguousarray(a.T)).to(DEV)


def _host(t: torch.Tensor) -> np.ndarray:
    """inverse of _dev_colmajor"""
    return t.cpu().numpy().T


def _ctx(w, max_mode=0):
    return hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=max_mode)


def _relmax(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


# ---------------------------------------------------------------------------------------------------- setup tables
@pytest.mark.parametrize("nb,a", [(2, 1.0), (5, 3.0), (37, 7.5), (50, 10.0), (100, 20.0), (151, 12.0)])
def test_mesh_matches_oracle(nb, a):
    w = make_workload(0, nch=2, nb=nb)
    ctx = hb.Context(2, nb, a, w.h2m, w.lval[:2], w.ethr[:2], max_mode=1 << hb.HPRMAT_FP64)
    r, fa = ctx.mesh()
    _, _, r_o, fa_o = oracle.mesh(nb, a)
    assert np.all(np.abs(r - r_o) <= 1 * np.spacing(r_o))
    assert np.all(np.abs(fa - fa_o) <= 1 * np.spacing(np.abs(fa_o)))
    ctx.destroy()


# ---------------------------------------------------------------------------------------------------- assembly
@pytest.mark.parametrize("cfg,nch,nb", [(0, None, None), (1, 8, 100), (1, 5, 37), (2, 1, 64), (3, 3, 130), (1, 33, 20)])
def test_assembly_parity(cfg, nch, nb):
    w = make_workload(cfg, nch=nch, nb=nb)
    ctx = _ctx(w, 1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    V = w.potential(r)
    E = float(w.energies[0])
    Cg = _host(ctx.get_matrix(E, torch.from_numpy(V).to(DEV)))
    Co = oracle.assemble(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, w.potential(oracle.mesh(w.nb, w.a)[2]))
    assert Cg.shape == Co.shape == (w.n, w.n)
    zero = Co == 0
    assert np.all(Cg[zero] == 0), "structural zeros must be exact"
    ulp = np.maximum(np.spacing(np.abs(Co.real)), np.spacing(np.abs(Co.imag)))
    assert np.all(np.abs(Cg.real - Co.real) <= 4 * np.spacing(np.abs(Co.real)) + 0 * ulp)
    assert np.all(np.abs(Cg.imag - Co.imag) <= 4 * np.spacing(np.abs(Co.imag)))
    assert np.abs(Cg - Cg.T).max() == 0.0 or _relmax(Cg, Cg.T) < 1e-15   # complex symmetric
    ctx.destroy()


# ---------------------------------------------------------------------------------------------------- raw GEMM / LU
@pytest.mark.parametrize("m,n,k", [(1, 1, 1), (32, 32, 32), (100, 50, 37), (257, 129, 65), (130, 33, 300), (1000, 333, 200),
                                   (5, 700, 3)])
def test_zgemm_matches_definition(m, n, k):
    rng = np.random.default_rng(m * 1000003 + n * 1009 + k)
    A = rng.uniform(-1, 1, (m, k)) + 1j * rng.uniform(-1, 1, (m, k))
    B = rng.uniform(-1, 1, (k, n)) + 1j * rng.uniform(-1, 1, (k, n))
    C0 = rng.uniform(-1, 1, (m, n)) + 1j * rng.uniform(-1, 1, (m, n))
    Cd = _dev_colmajor(C0)
    hb.hprmat_zgemm(m, n, k, -1.0, _dev_colmajor(A), m, _dev_colmajor(B), k, 1.0, Cd, m)
    ref = C0 - (A.astype(np.clongdouble) @ B.astype(np.clongdouble)).astype(np.complex128)
    assert np.abs(_host(Cd) - ref).max() <= 4 * (k + 2) * 2.0 ** -53 * 2.0 * max(1.0, np.abs(ref).max())


@pytest.mark.parametrize("algo", [3, 4])
def test_zgemm_both_real_decompositions(algo):
    """hprmat_zgemm_algo: the 3M kernel (three real products, imaginary part normwise accurate) and the 4M kernel against the
    definition in long double, with the NORMWISE bound (k + 4) 2^-52 (|A| |B|)_ij + 2^-52 |C0| that holds for both, on a
    ragged shape that spans several tiles of either kernel; and the switch reports what is in force."""
    prev = hb.hprmat_zgemm_algo()
    try:
        assert hb.hprmat_zgemm_algo(algo) == algo and hb.hprmat_zgemm_algo(0) == algo
        m, n, k = 333, 201, 150
        rng = np.random.default_rng(77 + algo)
        A = rng.normal(size=(m, k)) + 1j * rng.normal(size=(m, k))
        B = rng.normal(size=(k, n)) + 1j * rng.normal(size=(k, n))
        C0 = rng.normal(size=(m, n)) + 1j * rng.normal(size=(m, n))
        Cd = _dev_colmajor(C0)
        hb.hprmat_zgemm(m, n, k, -1.0, _dev_colmajor(A), m, _dev_colmajor(B), k, 1.0, Cd, m)
        ref = C0 - (A.astype(np.clongdouble) @ B.astype(np.clongdouble)).astype(np.complex128)
        absA, absB = np.abs(A.real) + np.abs(A.imag), np.abs(B.real) + np.abs(B.imag)
        bound = (k + 4) * 2.0 ** -52 * (absA @ absB) + 2.0 ** -52 * np.abs(C0)
        assert np.all(np.abs(_host(Cd) - ref) <= bound)
    finally:
        hb.hprmat_zgemm_algo(prev)


@pytest.mark.parametrize("n,nrhs", [(1, 1), (2, 3), (31, 1), (32, 5), (33, 2), (100, 7), (257, 4), (640, 64), (1500, 3)])
def test_zsolve_fp64_matches_oracle(n, nrhs):
    A = dense_test_matrix(n, nrhs, seed=7000 + n)
    B = np.asfortranarray(A @ np.ones((n, nrhs), dtype=np.complex128))       # x_exact = 1
    Xo = oracle.solve(A, B, mode=0, nrefine=2)
    assert np.abs(Xo - 1.0).max() < 1e-12                                    # the oracle itself reproduces x = 1
    Ad, Bd = _dev_colmajor(A), _dev_colmajor(B)
    ipiv, info = hb.hprmat_zsolve(n, nrhs, Ad, n, Bd, n)
    X = _host(Bd)
    assert info["status"] == 0
    assert _relmax(X, Xo) <= 1e-10
    # the factors left in A and the 1-based interchanges are a valid P A = L U (not compared with the oracle's: ties)
    LU = _host(Ad)
    L = np.tril(LU, -1) + np.eye(n)
    U = np.triu(LU)
    piv = ipiv.cpu().numpy() - 1
    assert piv.min() >= 0 and piv.max() < n and np.all(piv >= np.arange(n))
    PA = A.copy()
    for j in range(n):
        if piv[j] != j:
            PA[[j, piv[j]]] = PA[[piv[j], j]]
    assert np.abs(L @ U - PA).max() <= 50 * n * 2.0 ** -53 * np.abs(A).sum(1).max()
    assert np.abs(np.tril(LU, -1)).max() <= np.sqrt(2.0) + 1e-12             # partial pivoting on |re|+|im|


def test_zsolve_reports_singular():
    n = 64
    A = dense_test_matrix(n, 1, seed=99)
    A[:, 10] = 0.0
    Ad, Bd = _dev_colmajor(A), _dev_colmajor(np.ones((n, 1), dtype=np.complex128))
    with pytest.raises(hb.HprmatError) as e:
        hb.hprmat_zsolve(n, 1, Ad, n, Bd, n)
    assert e.value.code == hb.HPRMAT_ESINGULAR


def test_zsolve_empty():
    A = torch.zeros(1, dtype=torch.complex128, device=DEV)
    ipiv, info = hb.hprmat_zsolve(0, 0, A, 1, A, 1)
    assert info["status"] == 0


# ---------------------------------------------------------------------------------------------------- whole path, FP64
def _oracle_R(w, E, mode=0):
    r = oracle.mesh(w.nb, w.a)[2]
    return oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, w.potential(r), mode=mode, nrefine=2,
                          return_x=True)


@pytest.mark.parametrize("cfg,nch,nb", [(0, None, None), (0, 1, 50), (1, 8, 100), (1, 5, 37), (2, 16, 100), (3, 12, 64)])
def test_rmatrix_fp64_parity(cfg, nch, nb):
    w = make_workload(cfg, nch=nch, nb=nb)
    ctx = _ctx(w, 1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    V = torch.from_numpy(w.potential(r)).to(DEV)
    for E in w.energies[:2]:
        R, info = ctx.solve(float(E), V, hb.HPRMAT_FP64)
        Ro, Xo = _oracle_R(w, float(E))
        Rg = _host(R)
        assert info["status"] == 0
        assert _relmax(Rg, Ro) <= 1e-10, (info, _relmax(Rg, Ro))
        assert 0 <= info["backward_err"] <= 50 * w.n * 2.0 ** -53
        assert _relmax(_host(ctx.get_x()), Xo) <= 1e-10
        assert _relmax(Rg, Rg.T) <= 1e-10                                     # R = R^T since C = C^T
    ctx.destroy()


def test_rmatrix_fp64_host_entry_matches_device_entry():
    w = make_workload(0)
    ctx = _ctx(w, 1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    Vh = w.potential(r)
    R1, _ = ctx.solve(10.0, torch.from_numpy(Vh).to(DEV), hb.HPRMAT_FP64)
    R2, info = ctx.solve_host(10.0, Vh, hb.HPRMAT_FP64)
    assert np.array_equal(R1.cpu().numpy(), R2)
    assert info["ms_total"] > 0 and info["lu_tflops"] > 0
    ctx.destroy()


def test_rmatrix_no_info_path_is_asynchronous_and_equal():
    w = make_workload(1, nch=8, nb=100)
    ctx = _ctx(w, 1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    V = torch.from_numpy(w.potential(r)).to(DEV)
    R1, _ = ctx.solve(20.0, V, hb.HPRMAT_FP64, max_refine=1)
    R2, none = ctx.solve(20.0, V, hb.HPRMAT_FP64, max_refine=1, want_info=False)
    torch.cuda.synchronize()
    assert none is None
    assert _relmax(R2.cpu().numpy(), R1.cpu().numpy()) <= 1e-13
    ctx.destroy()


@pytest.mark.slow
def test_rmatrix_fp64_cfg1_full_size():
    """BASELINE.json configs[1] at full size (N = 6400), one energy; oracle in big-N mode (double accumulation in the
    factorisation, long-double residual refinement), which test_oracle_pins checks against the long-double mode."""
    w = make_workload(1)
    ctx = _ctx(w, 1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    V = torch.from_numpy(w.potential(r)).to(DEV)
    E = float(w.energies[3])
    R, info = ctx.solve(E, V, hb.HPRMAT_FP64)
    Ro, Xo = _oracle_R(w, E, mode=1)
    assert _relmax(_host(R), Ro) <= 1e-10, info
    assert 0 <= info["backward_err"] <= 50 * w.n * 2.0 ** -53
    ctx.destroy()


@pytest.mark.slow
@pytest.mark.parametrize("cfg", [3, 4])
def test_rmatrix_fp64_cfg3_headline_size_certificate(cfg):
    """BASELINE.json configs[3] (N = 25600) in the launch configuration bench.py times, and configs[4] (N = 51200: the 42 GB
    matrix in core; its first panels are taller than the register-resident kernel holds, so the shared-memory panel
    kernel runs too).  The full oracle needs ~10 / ~80 core-hours here, so correctness is certified from the oracle's
    long-double residual of the GPU solution."""
    w = make_workload(cfg)
    ctx = _ctx(w, 1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    V = torch.from_numpy(w.potential(r)).to(DEV)
    R, info = ctx.solve(30.0, V, hb.HPRMAT_FP64)
    X = _host(ctx.get_x())
    Rg = _host(R)
    c = certificate(w, 30.0, X, Rg)
    assert c["est"] <= 1e-10, (c, info)
    # the dropped second-order term O(||C^-1|| ||r||^2): bounded by the ORACLE's residual in the backward-error measure and
    # estimated explicitly (tests/certificate.py), neither taken from the library's own report
    assert c["backward_err"] <= 50 * w.n * 2.0 ** -53, c
    assert c["second"] <= 1e-12 and (c["contraction"] < 1.0 or c["second"] <= 1e-16), c
    assert 0 <= info["backward_err"] <= 50 * w.n * 2.0 ** -53
    assert _relmax(Rg, Rg.T) <= 1e-10
    # sampled outputs the oracle can compute one by one: R_c1c2 = (h2m/a) sum_i fa_i X[(c1,i),c2] from the GPU's X
    fa = oracle.mesh(w.nb, w.a)[3]
    for (c1, c2) in [(0, 0), (3, 200), (255, 255), (17, 4)]:
        assert abs(Rg[c1, c2] - (w.h2m / w.a) * np.dot(fa, X[c1 * w.nb:(c1 + 1) * w.nb, c2])) <= 1e-13 * np.abs(Rg).max()
    ctx.destroy()


# ---------------------------------------------------------------------------------------------------- FP64 factorisation variants
@pytest.mark.parametrize("cfg,nch,nb,E", [(0, None, None, 10.0), (1, 5, 37, 9.0), (1, 12, 100, 25.0), (3, 20, 130, 30.0)])
def test_both_fp64_factorisations_match_the_oracle(cfg, nch, nb, E):
    """hprmat_fp64_algo: 1 = LU of C - E I (the paper's Type 1), 2 = LU of the block-preconditioned S = K_d^-1 (C - E I)
    with verified diagonal pivots (default).  Both must meet the FP64 bar on R, X and the backward error of the ORIGINAL
    system."""
    w = make_workload(cfg, nch=nch, nb=nb)
    ctx = _ctx(w, 1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    V = torch.from_numpy(w.potential(r)).to(DEV)
    Ro, Xo = oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, w.potential(oracle.mesh(w.nb, w.a)[2]), return_x=True)
    default = hb.hprmat_fp64_algo()
    assert default == 2
    try:
        for algo in (1, 2):
            assert hb.hprmat_fp64_algo(algo) == algo
            R, info = ctx.solve(E, V, hb.HPRMAT_FP64)
            assert _relmax(_host(R), Ro) <= 1e-10, algo
            assert _relmax(_host(ctx.get_x()), Xo) <= 1e-9, algo
            assert 0 <= info["backward_err"] <= 50 * w.n * 2.0 ** -53, algo
            R2, none = ctx.solve(E, V, hb.HPRMAT_FP64, want_info=False)     # unsynchronised call, two unconditional steps
            torch.cuda.synchronize()
            assert none is None and _relmax(_host(R2), Ro) <= 1e-10, algo
    finally:
        hb.hprmat_fp64_algo(default)
    ctx.destroy()


def test_preconditioned_fp64_falls_back_to_pivoting_when_the_diagonal_is_refuted():
    """Couplings 300x the configs' make S pivot off the diagonal: the speculative FP64 panels are refuted and redone with
    partial pivoting (panel.cu); the result must still meet the FP64 bar, and equal the classic factorisation's."""
    w = make_workload(1, nch=12, nb=100)
    w.beta *= 300.0
    E = 20.0
    ctx = _ctx(w, 1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    V = torch.from_numpy(w.potential(r)).to(DEV)
    Ro = oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, w.potential(oracle.mesh(w.nb, w.a)[2]))
    R2, info2 = ctx.solve(E, V, hb.HPRMAT_FP64)
    R2 = _host(R2).copy()
    assert _relmax(R2, Ro) <= 1e-10 and info2["backward_err"] <= 50 * w.n * 2.0 ** -53
    assert info2["reserved"] > 0, "the diagonal-pivot speculation was expected to be refuted (info.reserved counts the panels)"
    # an unsynchronised call cannot fall back: it must say so through the device status word
    ctx.solve(E, V, hb.HPRMAT_FP64, want_info=False)
    assert ctx.last_status()[0] == hb.HPRMAT_EUNVERIFIED
    # ... and with the configs' own couplings it reports success
    w0 = make_workload(1, nch=12, nb=100)
    ctx.solve(E, torch.from_numpy(w0.potential(r)).to(DEV), hb.HPRMAT_FP64, want_info=False)
    assert ctx.last_status()[0] == hb.HPRMAT_OK
    try:
        hb.hprmat_fp64_algo(1)
        R1, _ = ctx.solve(E, V, hb.HPRMAT_FP64)
        assert _relmax(_host(R1), Ro) <= 1e-10
    finally:
        hb.hprmat_fp64_algo(2)
    ctx.destroy()


def test_preconditioned_fp64_falls_back_on_a_pole_of_an_uncoupled_channel():
    """Real potentials: at an eigenvalue of one diagonal block K_c (a pole of the UNCOUPLED channel) the preconditioner does
    not exist although the coupled matrix is regular; the synchronised FP64 call must notice and factor C - E I itself."""
    w = make_workload(0, nch=3, nb=40)
    w.W0 = 0.0
    ro = oracle.mesh(w.nb, w.a)[2]
    C0 = oracle.assemble(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, 0.0, w.potential(ro))
    ev = np.linalg.eigvalsh(C0[: w.nb, : w.nb].real)              # K_0 at E = 0: its eigenvalues are the poles of channel 0
    E = float(ev[np.argmin(np.abs(ev - 8.0))])
    ctx = _ctx(w, 1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    V = torch.from_numpy(w.potential(r)).to(DEV)
    Ro = oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, w.potential(ro))
    assert hb.hprmat_fp64_algo() == 2
    R, info = ctx.solve(E, V, hb.HPRMAT_FP64)
    assert info["status"] == hb.HPRMAT_OK
    assert _relmax(_host(R), Ro) <= 1e-10
    assert 0 <= info["backward_err"] <= 50 * w.n * 2.0 ** -53
    # a hair off the pole the preconditioner exists but is ill-conditioned
    for dE in (1e-9, 1e-6, 1e-3):
        Ro2 = oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E + dE, w.potential(ro))
        R2, info2 = ctx.solve(E + dE, V, hb.HPRMAT_FP64)
        assert info2["status"] == hb.HPRMAT_OK and _relmax(_host(R2), Ro2) <= 1e-10, dE
    ctx.destroy()
