"""Seeded synthetic inputs for the HPRMAT hot path (BASELINE.json `configs`).

This module is the ONLY code that both the CUDA path's callers (tests, bench.py) and the oracle's callers share.  It
holds none of the method's arithmetic: it only draws the channel tables (l_c, E_c, beta_cc') from a seeded PRNG and
evaluates the Woods-Saxon potential family at mesh radii that the caller passes in (the radii come from
`hprmat_mesh` on the GPU side and from `oracle.mesh` on the oracle side; tests assert they agree).

Recipe: diagonal V_cc(r) = -(V0 + i W0) f(r), f(r) = 1/(1 + exp((r - R)/a_ws)), the same for
every channel; coupling V_cc'(r) = beta_cc' * df/dr * (1 fm), beta symmetric ~ U[lo, hi] drawn in row-major order over
the upper triangle; thresholds E_0 = 0 and the remaining nch-1 ~ U[0, emax] sorted ascending; l_c = c mod 16.
The paper's own benchmark matrices are unspecified "synthetic test matrices with the same block structure"
(PAPER.md:354); these stand in for them.
"""
from dataclasses import dataclass, field

import numpy as np

H2M = 20.736 / 0.9          # hbar^2 / 2 mu in MeV fm^2, mu = 0.9 amu (BASELINE.json config 0)
A_WS = 0.65                 # Woods-Saxon diffuseness, fm
BASE_SEED = 251211590


@dataclass
class Workload:
    name: str
    nch: int
    nb: int
    a: float
    h2m: float
    lval: np.ndarray          # int32 [nch]
    ethr: np.ndarray          # float64 [nch], MeV
    energies: np.ndarray      # float64, MeV
    beta: np.ndarray          # float64 [nch, nch] symmetric, zero diagonal
    V0: float
    W0: float
    R_ws: float
    modes: tuple = field(default_factory=tuple)

    @property
    def n(self) -> int:
        return self.nch * self.nb

    def potential(self, r: np.ndarray) -> np.ndarray:
        """V[i, c2, c1] = V_{c1 c2}(r_i), complex128, shape (nb, nch, nch), C-order (c1 fastest)."""
        r = np.asarray(r, dtype=np.float64)
        assert r.shape == (self.nb,)
        u = (r - self.R_ws) / A_WS
        f = 1.0 / (1.0 + np.exp(u))
        df = -np.exp(u) / (A_WS * (1.0 + np.exp(u)) ** 2)
        V = np.empty((self.nb, self.nch, self.nch), dtype=np.complex128)
        V[:] = self.beta[None, :, :] * df[:, None, None]
        diag = -(self.V0 + 1j * self.W0) * f
        idx = np.arange(self.nch)
        V[:, idx, idx] = diag[:, None]
        return V


_TABLE = {
    # cfg: (nch, nb, a, A_mass or None->R given, R_ws, V0, W0, beta_lo, beta_hi, emax, energies, modes)
    0: dict(nch=4, nb=50, a=10.0, R_ws=3.0, V0=50.0, W0=10.0, blo=0.5, bhi=2.0, emax=None,
            energies=[10.0], modes=("fp64",)),
    1: dict(nch=64, nb=100, a=10.0, R_ws=1.2 * 40.0 ** (1.0 / 3.0), V0=50.0, W0=10.0, blo=0.1, bhi=1.0, emax=20.0,
            energies=list(np.linspace(5.0, 50.0, 10)), modes=("fp64", "mixed_refine")),
    2: dict(nch=128, nb=100, a=15.0, R_ws=1.2 * 58.0 ** (1.0 / 3.0), V0=50.0, W0=10.0, blo=0.1, bhi=1.0, emax=20.0,
            energies=list(np.linspace(5.0, 50.0, 5)), modes=("fp64", "mixed", "mixed_refine")),
    3: dict(nch=256, nb=100, a=20.0, R_ws=1.2 * 208.0 ** (1.0 / 3.0), V0=50.0, W0=20.0, blo=0.05, bhi=0.5, emax=40.0,
            energies=[30.0], modes=("fp64", "mixed_refine")),
    4: dict(nch=512, nb=100, a=20.0, R_ws=1.2 * 208.0 ** (1.0 / 3.0), V0=50.0, W0=20.0, blo=0.02, bhi=0.2, emax=40.0,
            energies=[30.0], modes=("mixed_refine", "fp64")),
}


def make_workload(cfg: int, nch: int | None = None, nb: int | None = None, seed: int | None = None) -> Workload:
    """BASELINE.json configs[cfg].  nch / nb may be overridden to make reduced-size cases of the same family."""
    t = dict(_TABLE[cfg])
    if nch is not None:
        t["nch"] = nch
    if nb is not None:
        t["nb"] = nb
    n = t["nch"]
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + cfg if seed is None else seed))
    beta = np.zeros((n, n))
    iu = np.triu_indices(n, k=1)                       # row-major over the upper triangle
    beta[iu] = rng.uniform(t["blo"], t["bhi"], size=len(iu[0]))
    beta = beta + beta.T
    if t["emax"] is None:
        ethr = np.arange(n, dtype=np.float64)          # config 0: thresholds 0,1,2,3 MeV
    else:
        ethr = np.concatenate([[0.0], np.sort(rng.uniform(0.0, t["emax"], size=n - 1))])
    lval = (np.arange(n) % 16).astype(np.int32)
    return Workload(name=f"cfg{cfg}" + ("" if nch is None and nb is None else f"_nch{n}_nb{t['nb']}"),
                    nch=n, nb=t["nb"], a=t["a"], h2m=H2M, lval=lval, ethr=ethr,
                    energies=np.asarray(t["energies"], dtype=np.float64), beta=beta, V0=t["V0"], W0=t["W0"],
                    R_ws=t["R_ws"], modes=t["modes"])


BETA_NL = 0.85   # fm, range of the non-locality (the Perey-Buck value)


def nonlocal_matrix(w: "Workload", r, xp=np):
    """Synthetic NON-LOCAL potential for SURVEY.md 8(f) row 4, Perey-Buck form built from the workload's local form factors:
        W_cc'(r, r') = U_cc'((r + r')/2) exp(-((r - r')/BETA_NL)^2) / (sqrt(pi) BETA_NL),
        U_cc = -(V0 + i W0) f(s),  U_cc' = beta_cc' df/ds (c != c'),
    returned as the N x N matrix of Lagrange-mesh matrix elements  a sqrt(lam_i lam_j) W_cc'(r_i, r_j)  (Gauss
    approximation; lam = Gauss-Legendre weights on (0,1) from numpy's leggauss), as an array of shape (nch, nb, nch, nb)
    indexed [c2, j, c1, i] -- its memory is the column-major N x N matrix with index c*nb + i.  Input generation only (no
    arithmetic of the method); xp = numpy, or torch for a device-resident build (r then a torch tensor on that device)."""
    lam = np.polynomial.legendre.leggauss(w.nb)[1] / 2.0
    if xp is np:
        r = np.asarray(r, dtype=np.float64)
        lamx, beta = lam, w.beta.astype(np.complex128)
    else:
        lamx = xp.as_tensor(lam, dtype=xp.float64, device=r.device)
        beta = xp.as_tensor(w.beta, dtype=xp.complex128, device=r.device)
    s = 0.5 * (r[:, None] + r[None, :])                     # [j, i]
    u = xp.exp((s - w.R_ws) / A_WS)
    f = 1.0 / (1.0 + u)
    df = -u / (A_WS * (1.0 + u) ** 2)
    g = xp.exp(-((r[:, None] - r[None, :]) / BETA_NL) ** 2) / (np.sqrt(np.pi) * BETA_NL)
    g = g * (w.a * xp.sqrt(lamx[:, None] * lamx[None, :]))
    Gdf = (g * df) + 0j
    Gf = (g * f) * (-(w.V0 + 1j * w.W0))
    shape = (w.nch, w.nb, w.nch, w.nb)
    W = np.empty(shape, dtype=np.complex128) if xp is np else xp.empty(shape, dtype=xp.complex128, device=r.device)
    W[...] = beta.T[:, None, :, None] * Gdf[None, :, None, :]   # [c2, j, c1, i] = beta[c1, c2] Gdf[j, i]; beta_cc = 0
    for c in range(w.nch):
        W[c, :, c, :] = Gf
    return W


def dense_test_matrix(n: int, nrhs: int, seed: int, shift: float | None = None):
    """Well-conditioned dense complex test system for the raw solve entry: A = G + shift*I with G_ij ~ U(-1,1) +
    i U(-1,1), x_exact = 1 (PAPER.md:563 manufactured solution), B = A @ 1 is left to the caller (it is arithmetic)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    A = rng.uniform(-1, 1, size=(n, n)) + 1j * rng.uniform(-1, 1, size=(n, n))
    A = np.asfortranarray(A)
    A[np.arange(n), np.arange(n)] += (np.sqrt(n) if shift is None else shift)
    return A
