"""The a-posteriori certificate (tests/certificate.py) checked against cases where the truth is known: the oracle's own
solution perturbed by a known amount.  CPU only."""
import numpy as np

import oracle
from certificate import anorm_inf, certificate
from paper_2512_11590_b200.workloads import make_workload


def _truth(w, E):
    r = oracle.mesh(w.nb, w.a)[2]
    return oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, E, w.potential(r), return_x=True)


def test_anorm_matches_the_dense_matrix():
    w = make_workload(1, nch=5, nb=23)
    r = oracle.mesh(w.nb, w.a)[2]
    V = w.potential(r)
    Cm = oracle.assemble(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, 17.0, V)
    assert abs(anorm_inf(w, 17.0, V) - np.abs(Cm).sum(axis=1).max()) <= 1e-12 * np.abs(Cm).sum(axis=1).max()


def test_certificate_sees_a_known_perturbation():
    """X~ = X + delta: the first-order term must reproduce R(X~) - R(X) to second order, and the second-order estimate must
    have the size of what is left."""
    w = make_workload(1, nch=6, nb=40)
    E = 12.0
    Ro, Xo = _truth(w, E)
    fa = oracle.mesh(w.nb, w.a)[3]
    rng = np.random.default_rng(3)
    for eps in (1e-4, 1e-8):
        Xp = Xo * (1.0 + eps * rng.normal(size=Xo.shape))
        Rp = oracle.contract(w.nch, w.nb, w.a, w.h2m, fa, Xp)
        true_err = np.abs(Rp - Ro).max() / np.abs(Ro).max()
        c = certificate(w, E, Xp, Rp, jacobi_steps=2)
        # ||R - R~||_max lies within ||first-order term||_max +- ||second-order term||_max
        assert abs(true_err - c["est"]) <= 2.0 * c["second"] + 1e-14, (eps, c, true_err)
        assert c["second"] < c["est"]
        assert c["contraction"] < 0.5
    c0 = certificate(w, E, Xo, Ro)
    assert c0["est"] <= 1e-13 and c0["backward_err"] <= 50 * w.n * 2.0 ** -53
