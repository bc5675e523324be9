#!/usr/bin/env python
"""Write the stored oracle R-matrices of the big configs ("a cfg 3/4 oracle run is done ONCE, its R
and wall time cached on disk keyed by a hash of the input arrays").

    python tests/golden/make_oracle_R.py --cfg 2 --energy 27.5 [--mode 1]

Calls ONLY oracle/ (the CPU checker) and the seeded input generator (paper_2512_11590_b200/workloads.py, which holds none of
the method's arithmetic); nothing here touches the CUDA path.  Output: tests/golden/oracle_R_cfg<k>_E<energy>.npz with
  R        nch x nch complex128, R[c1, c2] (PAPER.md:137 step 4, prefactor hbar^2/2 mu a per BASELINE.json)
  key      sha256 of (nch, nb, a, h2m, lval, ethr, energy, V) as laid out in input_key() -- the tests recompute it from
           the inputs they hand to the GPU and refuse the file on a mismatch
  seconds, threads, mode   wall time of orc_rmatrix (factor + solves + 2 long-double-residual refinement steps +
           contraction), OpenMP threads used, oracle mode (0 = long-double accumulation, 1 = "big-N": the O(N^3)
           factorisation accumulates in double, the long-double-residual refinement restores ~1e-15; the two modes are
           compared in tests/test_oracle_pins.py)
"""
import argparse
import hashlib
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def input_key(w, energy, V) -> str:
    h = hashlib.sha256()
    h.update(np.asarray([w.nch, w.nb], dtype=np.int64).tobytes())
    h.update(np.asarray([w.a, w.h2m, float(energy)], dtype=np.float64).tobytes())
    h.update(np.ascontiguousarray(w.lval, dtype=np.int32).tobytes())
    h.update(np.ascontiguousarray(w.ethr, dtype=np.float64).tobytes())
    h.update(np.ascontiguousarray(V, dtype=np.complex128).tobytes())
    return h.hexdigest()


def golden_path(cfg, energy) -> str:
    return os.path.join(HERE, f"oracle_R_cfg{cfg}_E{energy:g}.npz")


def main():
    import oracle
    from paper_2512_11590_b200.workloads import make_workload
    ap = argparse.ArgumentParser()
    ap.add_argument("--cfg", type=int, required=True)
    ap.add_argument("--energy", type=float, required=True)
    ap.add_argument("--mode", type=int, default=1, choices=[0, 1])
    args = ap.parse_args()
    w = make_workload(args.cfg)
    r = oracle.mesh(w.nb, w.a)[2]
    V = w.potential(r)
    R, sec = oracle.rmatrix(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, args.energy, V, mode=args.mode, nrefine=2,
                            return_seconds=True)
    out = golden_path(args.cfg, args.energy)
    np.savez_compressed(out, R=np.asarray(R), key=input_key(w, args.energy, V), seconds=sec, threads=oracle.num_threads(),
                        mode=args.mode, n=w.n)
    print(f"{out}: N={w.n}, mode={args.mode}, {sec:.1f} s on {oracle.num_threads()} threads")


if __name__ == "__main__":
    main()
