"""Parity of hprmat_collision (collision matrix of the open channels from R, neutral
and charged channels) with oracle.collision_matrix, through the C ABI.  Tolerance: max|U - U_orc| <= 1e-10 (|U| <= 1 for a unitary or
absorptive problem, so absolute = relative to the scale of U); the channel constants are evaluated independently on the
two sides (long double recurrences vs scipy.special)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2512_11590_b200 import binding as hb
from paper_2512_11590_b200.workloads import make_workload

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _dev_colmajor(a):
    return torch.from_numpy(np.ascontiguousarray(a.T)).to(DEV)


def _U_gpu(lval, ethr, E, h2m, a, R_dev, zze2=None):
    info = torch.zeros(1, dtype=torch.int32, device=DEV)
    U, nopen = hb.hprmat_collision(lval, ethr, E, h2m, a, R_dev, zze2=zze2, info_dev=info)
    torch.cuda.synchronize()
    assert int(info.item()) == 0
    return U.cpu().numpy().reshape(nopen, nopen).T, nopen


@pytest.mark.parametrize("cfg,nch,nb,E", [(0, None, None, 10.0),      # configs[0], all four channels open
                                          (0, None, None, 1.5),       # two open, two closed
                                          (0, None, None, 0.25),      # one open
                                          (1, 24, 40, 9.0),           # random thresholds in (0, 20): mixed open / closed
                                          (2, 70, 30, 12.0),          # nch spans two LU panels
                                          (3, 150, 20, 30.0)])        # nch > LEAF: recursion, GEMM updates
def test_collision_matrix_end_to_end_parity(cfg, nch, nb, E):
    """solve + matching on the GPU (R never leaves the device) against oracle.rmatrix + oracle.collision_matrix."""
    w = make_workload(cfg, nch=nch, nb=nb)
    ctx = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    R_dev, _ = ctx.solve(E, torch.from_numpy(w.potential(r)).to(DEV), mode=hb.HPRMAT_FP64)
    Ug, nopen = _U_gpu(w.lval, w.ethr, E, w.h2m, w.a, R_dev)
    Ro = oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, w.potential(oracle.mesh(w.nb, w.a)[2]))
    Uo, opn = oracle.collision_matrix(Ro, w.lval, w.ethr, E, w.h2m, w.a)
    assert nopen == len(opn) == int(np.sum(E > w.ethr))
    assert Ug.shape == Uo.shape
    assert np.abs(Ug - Uo).max() <= 1e-10
    assert np.abs(Ug - Ug.T).max() <= 1e-10                           # complex-symmetric problem: U = U^T
    assert np.linalg.svd(Ug, compute_uv=False).max() <= 1.0 + 1e-10   # absorptive potential: no flux is created
    ctx.destroy()


@pytest.mark.parametrize("l,x", [(0, 0.05), (0, 3.0), (1, 0.2), (3, 1.0), (7, 2.5), (12, 4.0), (15, 30.0), (2, 250.0),
                                 (15, 0.9)])
@pytest.mark.parametrize("closed_partner", [False, True])
def test_channel_functions_over_l_and_x(l, x, closed_partner):
    """Two channels, the same synthetic R on both sides: channel 0 open with k a = x and orbital momentum l (ranges from far
    below to far above the centrifugal barrier), channel 1 open or closed at the same |k| a.  Exercises the Bessel
    recurrences of the product against scipy's, including their derivatives."""
    a, h2m = 8.0, 20.736
    e0 = (x / a) ** 2 * h2m
    E = e0
    ethr = [0.0, 2.0 * e0 if closed_partner else 0.5 * e0]
    lval = [l, (l + 3) % 16]
    R = np.array([[0.31 + 0.02j, -0.07 + 0.01j], [-0.07 + 0.01j, 0.12 - 0.03j]])
    Ug, nopen = _U_gpu(lval, ethr, E, h2m, a, _dev_colmajor(R))
    Uo, opn = oracle.collision_matrix(R, lval, ethr, E, h2m, a)
    assert nopen == len(opn) == (1 if closed_partner else 2)
    assert np.abs(Ug - Uo).max() <= 1e-10 * max(1.0, np.abs(Uo).max())


def test_free_particles_give_the_unit_matrix():
    """V = 0 on the GPU path: U = 1 on the open channels (independent of the oracle)."""
    nb, a, h2m, E = 40, 8.0, 20.736, 6.0
    lval, ethr = [0, 2, 1, 3], [0.0, 1.5, 3.0, 9.0]
    ctx = hb.Context(4, nb, a, h2m, lval, ethr, max_mode=1 << hb.HPRMAT_FP64)
    R_dev, _ = ctx.solve(E, torch.zeros((nb, 4, 4), dtype=torch.complex128, device=DEV), mode=hb.HPRMAT_FP64)
    Ug, nopen = _U_gpu(lval, ethr, E, h2m, a, R_dev)
    assert nopen == 3
    assert np.abs(Ug - np.eye(3)).max() < 1e-9
    ctx.destroy()


def test_collision_edge_cases_and_errors():
    a, h2m = 8.0, 20.736
    R = _dev_colmajor(np.array([[0.3 + 0.0j, 0.1], [0.1, 0.2]]))
    # no open channel: nopen = 0, nothing written, OK
    U, nopen = hb.hprmat_collision([0, 1], [5.0, 6.0], 1.0, h2m, a, R)
    assert nopen == 0 and U.numel() == 0
    # a single open channel, nch = 1: U = (O - R rO')^-1 (I - R rI'), a pure phase for real R
    U1, n1 = _U_gpu([0], [0.0], 4.0, h2m, a, _dev_colmajor(np.array([[0.25 + 0.0j]])))
    assert n1 == 1 and abs(abs(U1[0, 0]) - 1.0) < 1e-13
    # energy exactly at a threshold
    with pytest.raises(hb.HprmatError) as e:
        hb.hprmat_collision([0, 1], [0.0, 3.0], 3.0, h2m, a, R)
    assert e.value.code == -6
    # negative orbital momentum
    with pytest.raises(hb.HprmatError) as e:
        hb.hprmat_collision([0, -1], [0.0, 3.0], 4.0, h2m, a, R)
    assert e.value.code == -3
    # workspace too small
    ws = torch.empty(256 + 64, dtype=torch.uint8, device=DEV)
    with pytest.raises(hb.HprmatError) as e:
        hb.hprmat_collision([0, 1], [0.0, 3.0], 4.0, h2m, a, R, ws=ws)
    assert e.value.code == hb.HPRMAT_ENOMEM
    assert hb.hprmat_collision_workspace_bytes(2) > 0 and hb.hprmat_collision_workspace_bytes(-1) == 0



def test_sub_barrier_channels_keep_unitarity_on_the_gpu():
    """Real potential, l = 12 at k a = 0.56: U^dagger U = 1 and U = U^T to rounding (oracle-independent), and parity."""
    from test_oracle_pins import _ws_potential
    nb, a, h2m, E = 40, 8.0, 20.736, 6.0
    lval, ethr = [0, 12, 1], [0.0, 5.9, 3.0]
    beta = np.array([[0.0, 12.0, 9.0], [12.0, 0.0, 15.0], [9.0, 15.0, 0.0]])
    V = _ws_potential(nb, a, 3, beta)
    ctx = hb.Context(3, nb, a, h2m, lval, ethr, max_mode=1 << hb.HPRMAT_FP64)
    R_dev, _ = ctx.solve(E, torch.from_numpy(V).to(DEV), mode=hb.HPRMAT_FP64)
    Ug, nopen = _U_gpu(lval, ethr, E, h2m, a, R_dev)
    assert nopen == 3
    assert np.abs(Ug.conj().T @ Ug - np.eye(3)).max() < 1e-11
    assert np.abs(Ug - Ug.T).max() < 1e-11
    Uo, _ = oracle.collision_matrix(oracle.rmatrix(3, nb, a, h2m, lval, ethr, E, V), lval, ethr, E, h2m, a)
    assert np.abs(Ug - Uo).max() <= 1e-10
    ctx.destroy()


# ---------------------------------------------------------------------------------------------------- charged channels
E2 = 1.43996


@pytest.mark.parametrize("cfg,nch,nb,E,z1z2", [(0, None, None, 10.0, 2.0),    # all open, eta ~ 0.3
                                               (0, None, None, 1.5, 8.0),     # two closed (Whittaker), eta ~ 3 under the barrier
                                               (1, 24, 40, 9.0, 20.0),        # mixed open / closed, l up to 15, eta up to ~ 10
                                               (2, 70, 30, 12.0, 6.0)])
def test_charged_collision_matrix_end_to_end_parity(cfg, nch, nb, E, z1z2):
    """Point-Coulomb repulsion added to the diagonal of the workload's potential; each channel gets its own charge product
    (z1z2 (1 + c/nch)) so that a per-channel indexing slip cannot cancel."""
    w = make_workload(cfg, nch=nch, nb=nb)
    zz = z1z2 * E2 * (1.0 + np.arange(w.nch) / w.nch)
    ctx = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    V = w.potential(r)
    idx = np.arange(w.nch)
    V[:, idx, idx] += zz[None, :] / r[:, None]
    R_dev, _ = ctx.solve(E, torch.from_numpy(V).to(DEV), mode=hb.HPRMAT_FP64)
    Ug, nopen = _U_gpu(w.lval, w.ethr, E, w.h2m, w.a, R_dev, zze2=zz)
    ro = oracle.mesh(w.nb, w.a)[2]
    Vo = w.potential(ro)
    Vo[:, idx, idx] += zz[None, :] / ro[:, None]
    Ro = oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, Vo)
    Uo, opn = oracle.collision_matrix(Ro, w.lval, w.ethr, E, w.h2m, w.a, zze2=zz)
    assert nopen == len(opn)
    assert np.abs(Ug - Uo).max() <= 1e-10
    assert np.abs(Ug - Ug.T).max() <= 1e-10
    ctx.destroy()


def test_pure_coulomb_potential_gives_the_unit_matrix_on_the_gpu():
    """V = Z1 Z2 e^2 / r only: U = 1 relative to Coulomb waves (oracle-independent; mesh convergence sets the 1e-8)."""
    nb, a, h2m, E = 60, 8.0, 20.736 / 0.9, 6.0
    lval, ethr = [0, 2, 1, 3], [0.0, 1.5, 3.0, 9.0]
    zz = np.array([2.0, 4.0, 1.0, 6.0]) * E2
    ctx = hb.Context(4, nb, a, h2m, lval, ethr, max_mode=1 << hb.HPRMAT_FP64)
    r, _ = ctx.mesh()
    V = np.zeros((nb, 4, 4), dtype=complex)
    for c in range(4):
        V[:, c, c] = zz[c] / r
    R_dev, _ = ctx.solve(E, torch.from_numpy(V).to(DEV), mode=hb.HPRMAT_FP64)
    Ug, nopen = _U_gpu(lval, ethr, E, h2m, a, R_dev, zze2=zz)
    assert nopen == 3
    assert np.abs(Ug - np.eye(3)).max() < 1e-8
    ctx.destroy()
