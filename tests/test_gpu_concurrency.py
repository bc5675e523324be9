"""include/hprmat.h: "one context per host thread / stream".  Two host threads, each with its own context on its own CUDA
stream, solve different problems at the same time (the ctypes calls release the GIL, so the library really runs on two host
threads and the GPU work of the two streams interleaves): every R must be bit-identical to the R of the same solve done alone.
What this exercises: per-context side streams and graph caches, the thread-local algorithm overrides, the pooled per-device
resources of the raw entries, the atomic launch counter.  Needs a B200 ("-m gpu")."""
import threading

import numpy as np
import pytest
import torch

from paper_2512_11590_b200 import binding as hb
from paper_2512_11590_b200.workloads import make_workload

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _solve_series(w, mode, energies, stream, fp64_algo=0):
    """a fresh context on `stream`, one solve per energy, returns the list of R as numpy arrays"""
    out = []
    with torch.cuda.stream(stream):
        ctx = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=1 << mode)
        if fp64_algo:
            ctx.set_option(hb.HPRMAT_OPT_FP64_ALGO, fp64_algo)
        r, _ = ctx.mesh()
        V = torch.from_numpy(w.potential(r)).to(DEV)
        for E in energies:
            R, info = ctx.solve(float(E), V, mode)
            assert info["status"] == hb.HPRMAT_OK, (E, info)
            out.append(R.cpu().numpy().copy())
        stream.synchronize()
        ctx.destroy()
    return out


CASES = [
    # (workload A, mode A, fp64_algo A), (workload B, mode B, fp64_algo B)
    ((2, 12, 100, hb.HPRMAT_MIXED_REFINE, 0), (1, 9, 64, hb.HPRMAT_FP64, 0)),
    ((1, 10, 100, hb.HPRMAT_FP64, 1), (2, 7, 100, hb.HPRMAT_FP64, 2)),          # pivoting LU next to verified-diagonal LU
    ((2, 16, 100, hb.HPRMAT_MIXED_REFINE, 0), (2, 11, 80, hb.HPRMAT_TYPE3, 0)),
]


@pytest.mark.parametrize("ca,cb", CASES)
def test_two_contexts_on_two_host_threads_and_streams(ca, cb):
    jobs = []
    for cfg, nch, nb, mode, algo in (ca, cb):
        w = make_workload(cfg, nch=nch, nb=nb)
        jobs.append((w, mode, [float(e) for e in list(w.energies)[:3]] * 2, algo))
    # alone, one after the other
    alone = [_solve_series(w, mode, es, torch.cuda.Stream(), algo) for (w, mode, es, algo) in jobs]
    # together
    results, errors = [None, None], []

    def work(k):
        try:
            torch.cuda.set_device(0)
            w, mode, es, algo = jobs[k]
            results[k] = _solve_series(w, mode, es, torch.cuda.Stream(), algo)
        except Exception as e:  # noqa: BLE001 - reported in the main thread
            errors.append((k, repr(e)))

    l0 = hb.hprmat_launch_count()
    threads = [threading.Thread(target=work, args=(k,)) for k in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=600)
    assert not errors, errors
    assert all(not t.is_alive() for t in threads)
    assert hb.hprmat_launch_count() > l0
    for k in range(2):
        assert len(results[k]) == len(alone[k])
        for Rt, Ra in zip(results[k], alone[k]):
            assert np.array_equal(Rt, Ra), (k, np.abs(Rt - Ra).max())


def test_raw_solves_from_two_host_threads():
    """hprmat_zsolve (no context: pooled per-device side resources) from two threads on two streams, FP64 and mixed."""
    def problem(n, nrhs, seed):
        g = np.random.default_rng(seed)
        A = g.normal(size=(n, n)) + 1j * g.normal(size=(n, n)) + 4.0 * np.sqrt(n) * np.eye(n)
        B = g.normal(size=(n, nrhs)) + 1j * g.normal(size=(n, nrhs))
        return A, B

    def run(A, B, mode, stream):
        n, nrhs = B.shape
        with torch.cuda.stream(stream):
            At = torch.from_numpy(np.ascontiguousarray(A.T)).to(DEV)
            Bt = torch.from_numpy(np.ascontiguousarray(B.T)).to(DEV)
            _, info = hb.hprmat_zsolve(n, nrhs, At, n, Bt, n, mode=mode)      # B <- X
            assert info["status"] == hb.HPRMAT_OK, info
            stream.synchronize()
            return Bt.cpu().numpy().T.copy()

    probs = [(problem(700, 9, 1), hb.HPRMAT_FP64), (problem(900, 17, 2), hb.HPRMAT_MIXED_REFINE)]
    alone = [run(A, B, mode, torch.cuda.Stream()) for ((A, B), mode) in probs]
    for (A, B), X in zip([p[0] for p in probs], alone):
        assert np.abs(A @ X - B).max() <= 1e-10 * np.abs(B).max() * A.shape[0]
    results, errors = [None, None], []

    def work(k):
        try:
            torch.cuda.set_device(0)
            (A, B), mode = probs[k]
            for _ in range(3):
                results[k] = run(A, B, mode, torch.cuda.Stream())
        except Exception as e:  # noqa: BLE001
            errors.append((k, repr(e)))

    threads = [threading.Thread(target=work, args=(k,)) for k in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=600)
    assert not errors, errors
    for k in range(2):
        assert np.array_equal(results[k], alone[k]), (k, np.abs(results[k] - alone[k]).max())


@pytest.mark.parametrize("mode", [hb.HPRMAT_MIXED_REFINE, hb.HPRMAT_FP64])
def test_interleaved_scan_equals_the_sequential_scan(mode):
    """scan.interleaved_scan: the energies of a scan handed out to two contexts on two threads / streams; every R-matrix
    bit-identical to the one-context scan (each solve is one hprmat_solve, whichever context takes it)."""
    from paper_2512_11590_b200 import scan
    w = make_workload(2, nch=14, nb=100)
    energies = [float(e) for e in w.energies] + [float(e) + 0.37 for e in w.energies]
    R1, infos1, _ = scan.interleaved_scan(w, energies, mode, nctx=1)
    R2, infos2, _ = scan.interleaved_scan(w, energies, mode, nctx=2)
    assert all(i["status"] == hb.HPRMAT_OK for i in infos1 + infos2)
    assert np.array_equal(R1, R2)
    assert np.abs(R1).max() > 0

