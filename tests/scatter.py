"""Test-side scattering helpers (neutral case, eta = 0): Riccati-Bessel functions, the closed-form R-matrix of a
constant potential, and the collision matrix S from R.  Used only to PIN the oracle ("matching to
asymptotic solutions"); none of this is on the hot path and none of it is shared with oracle/ or the CUDA path.

F_l(x) = x j_l(x), G_l(x) = -x y_l(x), O = G + iF, I = G - iF.
Regular solution of a constant potential -V0 in partial wave l: u(r) = F_l(K r), K = sqrt((E + V0)/h2m), so
R = u(a) / (a u'(a)) = F_l(Ka) / (Ka F_l'(Ka)).
"""
import mpmath as mp
import numpy as np
from scipy.special import spherical_jn, spherical_yn


def F(l, x):
    return x * spherical_jn(l, x)


def dF(l, x):
    return spherical_jn(l, x) + x * spherical_jn(l, x, derivative=True)


def G(l, x):
    return -x * spherical_yn(l, x)


def dG(l, x):
    return -spherical_yn(l, x) - x * spherical_yn(l, x, derivative=True)


def R_constant_potential(l: int, K: complex, a: float) -> complex:
    """F_l(Ka)/(Ka F_l'(Ka)) for real or complex K (complex K: closed channel or absorptive well), via mpmath."""
    mp.mp.dps = 40
    z = mp.mpc(K) * a
    nu = l + mp.mpf(1) / 2
    f = lambda t: mp.sqrt(mp.pi * t / 2) * mp.besselj(nu, t)      # t j_l(t)
    val = f(z) / (z * mp.diff(f, z))
    return complex(val)


def smatrix(R: np.ndarray, lval, k: np.ndarray, a: float) -> np.ndarray:
    """S = (Z^O)^-1 Z^I,  Z^O_cc' = (k_c' a)^-1/2 [O_c(k_c a) delta_cc' - k_c' a R_cc' O'_c'(k_c' a)]  (all channels
    open).  Descouvemont & Baye, Rep. Prog. Phys. 73 (2010) Eq. (3.27)-(3.29) -- the paper's ref. [2]."""
    nch = len(lval)
    x = np.asarray(k, dtype=float) * a
    O = np.array([G(l, xx) + 1j * F(l, xx) for l, xx in zip(lval, x)])
    dO = np.array([dG(l, xx) + 1j * dF(l, xx) for l, xx in zip(lval, x)])
    ZO = (np.diag(O) - R * (x * dO)[None, :]) / np.sqrt(x)[None, :]
    ZI = (np.diag(O.conj()) - R * (x * dO.conj())[None, :]) / np.sqrt(x)[None, :]
    return np.linalg.solve(ZO, ZI)
