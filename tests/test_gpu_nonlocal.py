"""Parity of hprmat_solve_nonlocal (non-local potentials, every block of the matrix full;
PAPER.md:99, 155) with oracle.rmatrix_nonlocal, through the C ABI.  Tolerances as for the local path (north_star):
FP64 and mixed+refine max|R - R_orc| / max|R_orc| <= 1e-10, mixed without refinement <= 1e-3, backward error
<= 50 N 2^-53 wherever refinement ran."""
import itertools

import numpy as np
import pytest
import torch

import oracle
from paper_2512_11590_b200 import binding as hb
from paper_2512_11590_b200.workloads import make_workload, nonlocal_matrix

pytestmark = pytest.mark.gpu
DEV = "cuda"
H2M = 20.736 / 0.9


def _relmax(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


@pytest.mark.parametrize("cfg,nch,nb,E", [(0, None, None, 10.0),      # configs[0]
                                          (1, 7, 37, 9.0),            # ragged: N = 259
                                          (1, 8, 100, 25.0),          # N = 800: several LEAF blocks
                                          (2, 12, 100, 12.0),         # N = 1200: one 1024 solve block + ragged rest
                                          (3, 20, 130, 30.0)])        # N = 2600
def test_nonlocal_rmatrix_parity(cfg, nch, nb, E):
    w = make_workload(cfg, nch=nch, nb=nb)
    ctx = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    W_dev = torch.from_numpy(nonlocal_matrix(w, r)).to(DEV)                   # memory = column-major N x N
    R_dev, info = ctx.solve_nonlocal(E, W_dev)
    Rg = R_dev.cpu().numpy().T
    Wo = nonlocal_matrix(w, oracle.mesh(w.nb, w.a)[2]).reshape(w.n, w.n).T
    Ro, Xo = oracle.rmatrix_nonlocal(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, Wo, return_x=True)
    assert _relmax(Rg, Ro) <= 1e-10
    assert 0 <= info["backward_err"] <= 50 * w.n * 2.0 ** -53
    assert info["status"] == hb.HPRMAT_OK and info["refine_steps"] >= 1
    assert _relmax(Rg, Rg.T) <= 1e-10                                         # complex-symmetric W: R = R^T
    Xg = ctx.get_x().cpu().numpy().T
    assert _relmax(Xg, Xo) <= 1e-8
    ctx.destroy()


def test_local_potential_through_the_nonlocal_entry_and_padded_ldw():
    """W = V(r_i) delta_ij block-wise must give what hprmat_solve gives (oracle-independent); ldw > N is honoured."""
    w = make_workload(1, nch=6, nb=50)
    E = 15.0
    ctx = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    V = w.potential(r)
    ldw = w.n + 5
    Wp = np.full((w.n, ldw), 7.0 + 7.0j)                                      # [col, row]; the padding rows hold garbage
    Wp[:, : w.n] = 0.0
    for c1, c2 in itertools.product(range(w.nch), range(w.nch)):
        Wp[c2 * w.nb + np.arange(w.nb), c1 * w.nb + np.arange(w.nb)] = V[:, c2, c1]
    Rn, info = ctx.solve_nonlocal(E, torch.from_numpy(Wp).to(DEV), ldw=ldw)
    Rn = Rn.cpu().numpy().T.copy()
    Rl, _ = ctx.solve(E, torch.from_numpy(V).to(DEV), mode=hb.HPRMAT_FP64)
    assert _relmax(Rn, Rl.cpu().numpy().T) <= 1e-11
    assert info["backward_err"] <= 50 * w.n * 2.0 ** -53
    ctx.destroy()


@pytest.mark.parametrize("E", [0.5, 5.0, 30.0])
def test_separable_potential_phase_shift_on_the_gpu(E):
    """Rank-one kernel -lambda exp(-beta (r + r')): closed-form s-wave phase shift (derivation in
    tests/test_oracle_pins.py::test_separable_potential_has_the_analytic_phase_shift); solve + matching on the device."""
    nb, a, beta, lam0 = 60, 12.0, 2.0, 400.0
    ctx = hb.Context(1, nb, a, H2M, [0], [0.0], max_mode=1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    lam = np.polynomial.legendre.leggauss(nb)[1] / 2.0
    W = -lam0 * a * np.sqrt(np.outer(lam, lam)) * np.exp(-beta * (r[:, None] + r[None, :])) + 0j
    R_dev, _ = ctx.solve_nonlocal(E, torch.from_numpy(np.ascontiguousarray(W.T)).to(DEV))
    U, nopen = hb.hprmat_collision([0], [0.0], E, H2M, a, R_dev)
    k = np.sqrt(E / H2M)
    Lam = lam0 / H2M
    tan_d = Lam * k / ((beta ** 2 + k ** 2) ** 2 + Lam * (k ** 2 - beta ** 2) / (2 * beta))
    S_exact = (1 + 1j * tan_d) / (1 - 1j * tan_d)
    assert nopen == 1 and abs(U.cpu().numpy()[0] - S_exact) < 1e-8
    ctx.destroy()


def test_nonlocal_argument_errors_and_unsynchronised_call():
    w = make_workload(0)
    ctx = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=0)
    r, _ = ctx.mesh()
    W_dev = torch.from_numpy(nonlocal_matrix(w, r)).to(DEV)
    with pytest.raises(hb.HprmatError) as e:
        ctx.solve_nonlocal(10.0, W_dev, mode=17)
    assert e.value.code == -5
    with pytest.raises(hb.HprmatError) as e:
        hb._check(hb.lib().hprmat_solve_nonlocal(ctx._h, hb.C.c_double(10.0), hb._dev(W_dev), hb.C.c_long(w.n - 1),
                                                 hb.C.c_int(hb.HPRMAT_FP64), hb.C.c_int(-1), hb.C.c_double(0.0),
                                                 hb._dev(W_dev), None), "hprmat_solve_nonlocal")
    assert e.value.code == -4
    # info == NULL: enqueue only; the result equals the synchronised call
    R1, _ = ctx.solve_nonlocal(10.0, W_dev)
    R1 = R1.clone()
    R2, none = ctx.solve_nonlocal(10.0, W_dev, want_info=False)
    torch.cuda.synchronize()
    assert none is None and _relmax(R2.cpu().numpy(), R1.cpu().numpy()) <= 1e-12
    # a context without the FP64 buffers refuses the FP64 mode (and the other way round)
    ctx2 = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=1 << hb.HPRMAT_MIXED_REFINE)
    with pytest.raises(hb.HprmatError) as e:
        ctx2.solve_nonlocal(10.0, W_dev)
    assert e.value.code == -5
    ctx3 = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=1 << hb.HPRMAT_FP64)
    with pytest.raises(hb.HprmatError) as e:
        ctx3.solve_nonlocal(10.0, W_dev, mode=hb.HPRMAT_MIXED_REFINE)
    assert e.value.code == -5
    ctx3.destroy()
    ctx.destroy()
    ctx2.destroy()


def test_nonlocal_full_size_properties():
    """BASELINE.json configs[3] (Nc = 256, Nb = 100, N = 25600) with the non-local workload built on the device; the oracle
    cannot reach this size, so what holds at any size is checked: backward error, symmetry of R, convergence status, and the
    collision matrix of the absorptive problem (singular values <= 1, U = U^T)."""
    w = make_workload(3)
    E = float(w.energies[0])
    ctx = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    W_dev = nonlocal_matrix(w, torch.from_numpy(r).to(DEV), xp=torch)
    assert W_dev.is_contiguous() and W_dev.numel() == w.n * w.n
    R_dev, info = ctx.solve_nonlocal(E, W_dev)
    assert info["status"] == hb.HPRMAT_OK
    assert 0 <= info["backward_err"] <= 50 * w.n * 2.0 ** -53
    Rg = R_dev.cpu().numpy().T
    assert np.all(np.isfinite(Rg.real)) and np.all(np.isfinite(Rg.imag))
    assert _relmax(Rg, Rg.T) <= 1e-10
    U, nopen = hb.hprmat_collision(w.lval, w.ethr, E, w.h2m, w.a, R_dev)
    Ug = U.cpu().numpy().reshape(nopen, nopen).T
    assert nopen == int(np.sum(E > w.ethr))
    assert np.abs(Ug - Ug.T).max() <= 1e-10
    assert np.linalg.svd(Ug, compute_uv=False).max() <= 1.0 + 1e-10
    print(f"non-local cfg3: lu {info['ms_lu']:.1f} ms, total {info['ms_total']:.1f} ms, backward error {info['backward_err']:.2e}, "
          f"refine steps {info['refine_steps']}")
    ctx.destroy()
    del W_dev
    torch.cuda.empty_cache()


# ---------------------------------------------------------------------------------------------------- mixed modes
@pytest.mark.parametrize("cfg,nch,nb,E", [(0, None, None, 10.0), (1, 7, 37, 9.0), (1, 8, 100, 25.0), (2, 12, 100, 12.0),
                                          (3, 20, 130, 30.0)])
def test_nonlocal_mixed_modes_parity(cfg, nch, nb, E):
    """TF32 factors of S = K_d^-1 (K + W) (full blocks) with and without FP64 refinement."""
    w = make_workload(cfg, nch=nch, nb=nb)
    ctx = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr,
                     max_mode=(1 << hb.HPRMAT_MIXED) | (1 << hb.HPRMAT_MIXED_REFINE))
    r, _ = ctx.mesh()
    W_dev = torch.from_numpy(nonlocal_matrix(w, r)).to(DEV)
    Wo = nonlocal_matrix(w, oracle.mesh(w.nb, w.a)[2]).reshape(w.n, w.n).T
    Ro = oracle.rmatrix_nonlocal(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, Wo)
    R1, info1 = ctx.solve_nonlocal(E, W_dev, mode=hb.HPRMAT_MIXED)
    assert info1["status"] == hb.HPRMAT_OK and info1["refine_steps"] == 0
    assert _relmax(R1.cpu().numpy().T, Ro) <= 1e-3
    R2, info2 = ctx.solve_nonlocal(E, W_dev, mode=hb.HPRMAT_MIXED_REFINE)
    assert info2["status"] == hb.HPRMAT_OK and 1 <= info2["refine_steps"] <= 5
    assert _relmax(R2.cpu().numpy().T, Ro) <= 1e-10
    assert 0 <= info2["backward_err"] <= 50 * w.n * 2.0 ** -53
    ctx.destroy()


def test_nonlocal_mixed_full_size_properties():
    """configs[3] size, mixed + refinement: converged status, backward error, R = R^T, and agreement with the FP64 mode
    of the same entry (two different factorisations of two different matrices, S and C) to 1e-9."""
    w = make_workload(3)
    E = float(w.energies[0])
    ctx = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=0)
    r, _ = ctx.mesh()
    W_dev = nonlocal_matrix(w, torch.from_numpy(r).to(DEV), xp=torch)
    Rm, info = ctx.solve_nonlocal(E, W_dev, mode=hb.HPRMAT_MIXED_REFINE)
    Rm = Rm.cpu().numpy().T.copy()
    assert info["status"] == hb.HPRMAT_OK
    assert 0 <= info["backward_err"] <= 50 * w.n * 2.0 ** -53
    assert _relmax(Rm, Rm.T) <= 1e-10
    Rf, info_f = ctx.solve_nonlocal(E, W_dev, mode=hb.HPRMAT_FP64)
    assert _relmax(Rm, Rf.cpu().numpy().T) <= 1e-9
    print(f"non-local cfg3 mixed+refine: assemble {info['ms_assemble']:.1f} ms, lu {info['ms_lu']:.1f} ms, total "
          f"{info['ms_total']:.1f} ms, {info['refine_steps']} steps, backward error {info['backward_err']:.2e}; fp64 total "
          f"{info_f['ms_total']:.1f} ms")
    ctx.destroy()
    del W_dev
    torch.cuda.empty_cache()
