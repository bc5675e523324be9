"""Host logic of the matching step (hprmat_channel_functions of include/hprmat.h: no CUDA call, so it runs in the CPU
suite): the long-double Bessel recurrences / Steed continued fractions of the product against the oracle's mpmath values,
and against what the mathematics fixes (Wronskian, closed forms)."""
import itertools

import numpy as np
import pytest

from oracle.oracle import _coulomb_channel
from paper_2512_11590_b200 import binding as hb


def _rel(g, o):
    return max(abs(a - b) / max(abs(b), 1e-300) for a, b in zip(g, o))


@pytest.mark.parametrize("eta", [0.0, 0.01, 0.3, 2.5, 8.0, 20.0, -0.5, -3.0])
def test_open_channel_functions_match_the_oracle(eta):
    for l, x in itertools.product([0, 3, 15], [0.05, 0.7, 4.0, 25.0]):
        g = hb.hprmat_channel_functions(l, eta, x, True)
        o = _coulomb_channel(l, eta, x, True)
        assert _rel(g, o) < 1e-12, (l, eta, x, g, o)


@pytest.mark.parametrize("eta", [0.0, 0.3, 2.5, 8.0, -3.0])
def test_closed_channel_logarithmic_derivative_matches_the_oracle(eta):
    for l, x in itertools.product([0, 1, 4, 15], [0.05, 0.7, 4.0, 25.0, 200.0]):
        g = hb.hprmat_channel_functions(l, eta, x, False)
        o = _coulomb_channel(l, eta, x, False)
        assert g[:3] == (0.0, 0.0, 1.0)
        assert abs(g[3] - o[3]) <= 1e-13 * max(1.0, abs(o[3])), (l, eta, x, g, o)


def test_wronskian_and_closed_forms():
    # F'G - FG' = 1 for every (l, eta, x), including far under the barrier where F ~ 1e-30
    for l, eta, x in itertools.product([0, 2, 9, 15], [0.0, 0.2, 3.0, 12.0, -2.0], [0.01, 0.3, 2.0, 17.0, 300.0]):
        F, xdF, G, xdG = hb.hprmat_channel_functions(l, eta, x, True)
        assert abs((xdF * G - F * xdG) / x - 1.0) < 1e-13, (l, eta, x)
    # eta = 0, l = 0: sin, cos, exp(-x);  l = 1: W = exp(-x)(1 + 1/x)
    for x in [0.01, 0.5, 3.0, 40.0]:
        F, xdF, G, xdG = hb.hprmat_channel_functions(0, 0.0, x, True)
        assert abs(F - np.sin(x)) < 1e-15 and abs(G - np.cos(x)) < 1e-15
        assert abs(xdF - x * np.cos(x)) < 1e-15 * max(1, x) and abs(xdG + x * np.sin(x)) < 1e-15 * max(1, x)
        assert hb.hprmat_channel_functions(0, 0.0, x, False)[3] == pytest.approx(-x, rel=1e-15)
        assert hb.hprmat_channel_functions(1, 0.0, x, False)[3] == pytest.approx(-x - 1.0 / (x + 1.0), rel=1e-15)
    # a terminating continued fraction: l = 1, eta = -3, x = 4 gives x W'/W = 0 exactly
    assert hb.hprmat_channel_functions(1, -3.0, 4.0, False)[3] == 0.0


def test_argument_errors():
    for args, code in [((-1, 0.0, 1.0), -1), ((0, float("nan"), 1.0), -2), ((0, 0.0, 0.0), -3), ((0, 0.0, -1.0), -3),
                       ((0, 0.0, float("inf")), -3)]:
        with pytest.raises(hb.HprmatError) as e:
            hb.hprmat_channel_functions(*args)
        assert e.value.code == code
