"""Propagation over sub-intervals on the GPU (hprmat_setup_sector / hprmat_solve_sector / hprmat_propagate; SURVEY.md 8(f) row 4,
PAPER.md:53, 327; reading R16) against the oracle (oracle.sector_tables / sector_matrices / propagate), which is
pinned to closed forms in tests/test_oracle_pins.py.  Needs a B200 ("-m gpu")."""
import numpy as np
import pytest
import torch

import oracle
from paper_2512_11590_b200 import binding as hb
from paper_2512_11590_b200.workloads import make_workload

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _relmax(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


@pytest.mark.parametrize("nb,a_lo,a_hi", [(8, 1.0, 2.5), (37, 4.5, 10.0), (100, 9.0, 20.0)])
def test_sector_mesh_matches_oracle(nb, a_lo, a_hi):
    w = make_workload(0, nch=2, nb=nb)
    ctx = hb.Context.sector(2, nb, a_lo, a_hi, w.h2m, w.lval[:2], w.ethr[:2], max_mode=1 << hb.HPRMAT_FP64)
    r, fa = ctx.mesh()
    ro, _, faR, _ = oracle.sector_tables(nb, a_lo, a_hi)
    assert np.all(np.abs(r - ro) <= 2 * np.spacing(ro))
    assert np.all(np.abs(fa - faR) <= 1e-13 * np.abs(faR).max())
    ctx.destroy()


CASES = [(0, None, 50, 0.45), (1, 6, 60, 0.5), (2, 9, 100, 0.6), (1, 3, 33, 0.3)]


@pytest.mark.parametrize("cfg,nch,nb,frac", CASES)
@pytest.mark.parametrize("mode,tol", [(hb.HPRMAT_FP64, 1e-10), (hb.HPRMAT_MIXED_REFINE, 1e-10), (hb.HPRMAT_MIXED, 1e-3)])
def test_sector_matrices_and_propagated_rmatrix_match_oracle(cfg, nch, nb, frac, mode, tol):
    """Two sub-intervals (0, a_1), (a_1, a): R(a_1) from the ordinary path, the four sector matrices of (a_1, a), the propagated
    R(a) -- each against the oracle within the mode's tolerance; and the propagated R(a) against the GPU's own single-interval
    R(a) to the discretisation level."""
    w = make_workload(cfg, nch=nch, nb=nb)
    E = float(w.energies[0])
    a1 = frac * w.a
    mm = 1 << mode
    c1 = hb.Context(w.nch, w.nb, a1, w.h2m, w.lval, w.ethr, max_mode=mm)
    r1, _ = c1.mesh()
    R1, info1 = c1.solve(E, torch.from_numpy(w.potential(r1)).to(DEV), mode)
    assert info1["status"] == 0
    cs = hb.Context.sector(w.nch, w.nb, a1, w.a, w.h2m, w.lval, w.ethr, max_mode=mm)
    rs, _ = cs.mesh()
    Rsec, info = cs.solve_sector(E, torch.from_numpy(w.potential(rs)).to(DEV), mode)
    assert info["status"] == 0
    R2 = hb.hprmat_propagate(a1, w.a, R1, Rsec)
    # oracle
    ro1 = oracle.mesh(w.nb, a1)[2]
    R1o = oracle.rmatrix(w.nch, w.nb, a1, w.h2m, w.lval, w.ethr, E, w.potential(ro1))
    ros = oracle.sector_tables(w.nb, a1, w.a)[0]
    So = oracle.sector_matrices(w.nch, w.nb, a1, w.a, w.h2m, w.lval, w.ethr, E, w.potential(ros))
    R2o = oracle.propagate(a1, w.a, R1o, So)
    Sg = Rsec.cpu().numpy()
    scale = max(np.abs(So[a][b]).max() for a in range(2) for b in range(2))
    for k, (a, b) in enumerate([(0, 0), (0, 1), (1, 0), (1, 1)]):
        assert np.abs(Sg[k].T - So[a][b]).max() <= tol * scale, (k, info)
    assert _relmax(R2.cpu().numpy().T, R2o) <= 10 * tol, info
    if mode != hb.HPRMAT_MIXED:
        # (the mixed refinement stops at an estimated error of 1e-12, not at the last bit: floor the bound's N for tiny systems)
        assert 0 <= info["backward_err"] <= 50 * max(w.n, 1000) * 2.0 ** -53
        cf = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=mm)
        rf, _ = cf.mesh()
        Rf, _ = cf.solve(E, torch.from_numpy(w.potential(rf)).to(DEV), mode)
        assert _relmax(R2.cpu().numpy(), Rf.cpu().numpy()) <= 1e-6       # two discretisations of the same R(a)
        cf.destroy()
    c1.destroy()
    cs.destroy()


def test_three_sub_intervals_chain():
    """ns = 3: (0, a/3), (a/3, 2a/3), (2a/3, a) chained through hprmat_propagate, against the oracle's chain."""
    w = make_workload(0, nb=40)
    E, nb = 10.0, 40
    cuts = [w.a / 3, 2 * w.a / 3, w.a]
    c1 = hb.Context(w.nch, nb, cuts[0], w.h2m, w.lval, w.ethr, max_mode=1 << hb.HPRMAT_FP64)
    r1, _ = c1.mesh()
    R, _ = c1.solve(E, torch.from_numpy(w.potential(r1)).to(DEV), hb.HPRMAT_FP64)
    Ro = oracle.rmatrix(w.nch, nb, cuts[0], w.h2m, w.lval, w.ethr, E, w.potential(oracle.mesh(nb, cuts[0])[2]))
    for lo, hi in zip(cuts[:-1], cuts[1:]):
        cs = hb.Context.sector(w.nch, nb, lo, hi, w.h2m, w.lval, w.ethr, max_mode=1 << hb.HPRMAT_FP64)
        rs, _ = cs.mesh()
        Rsec, info = cs.solve_sector(E, torch.from_numpy(w.potential(rs)).to(DEV), hb.HPRMAT_FP64)
        R = hb.hprmat_propagate(lo, hi, R, Rsec)
        ros = oracle.sector_tables(nb, lo, hi)[0]
        Ro = oracle.propagate(lo, hi, Ro, oracle.sector_matrices(w.nch, nb, lo, hi, w.h2m, w.lval, w.ethr, E, w.potential(ros)))
        cs.destroy()
    assert _relmax(R.cpu().numpy().T, Ro) <= 1e-9
    c1.destroy()
