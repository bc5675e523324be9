"""Energy-scan bookkeeping: across N > 1 GPUs (replicas only) and, on one GPU, across several
contexts whose factorisations interleave (interleaved_scan).

One LU does not shard, the energy scan does: rank r of `world` takes the energies r, r + world, r + 2 world, ... of the
scan, solves them with its own context on its own GPU, and the Nc x Nc R-matrices are gathered at the end.  There is no
data-path collective; torch.distributed (nccl on GPUs, gloo in the CPU tests) only carries the gather, the barrier and the
max of the per-rank device times.  Nothing of the method's arithmetic lives here.
"""
from typing import Dict, List, Sequence

import numpy as np
import torch
import torch.distributed as dist


def shard_indices(n_energies: int, rank: int, world: int) -> List[int]:
    """Indices of the scan's energies handled by `rank` (round robin, so every rank gets a similar mix)."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    return list(range(rank, n_energies, world))


def bench_energy(energies: Sequence[float], rank: int) -> float:
    """The single energy a bench replica solves: the rank-th point of the scan, continued at the scan's spacing (or by
    0.5 MeV for a one-point scan) when there are more ranks than points."""
    e = [float(x) for x in energies]
    if rank < len(e):
        return e[rank]
    step = (e[-1] - e[0]) / (len(e) - 1) if len(e) > 1 else 0.5
    return e[-1] + step * (rank - len(e) + 1)


def max_over_ranks(value: float, device="cpu") -> float:
    """MAX over ranks of a per-rank scalar (the timing rule: a multi-GPU number is the slowest rank's device time)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_rmatrices(local: Dict[int, np.ndarray], n_energies: int, nch: int, device="cpu") -> np.ndarray:
    """All ranks' R-matrices in scan order: (n_energies, nch, nch) complex128 on every rank.  `local` maps scan index ->
    nch x nch array for the indices of shard_indices(...)."""
    out = torch.zeros((n_energies, nch, nch, 2), dtype=torch.float64, device=device)
    for i, R in local.items():
        R = np.asarray(R, dtype=np.complex128)
        if R.shape != (nch, nch):
            raise ValueError("R-matrix of the wrong shape")
        out[i, :, :, 0] = torch.from_numpy(np.ascontiguousarray(R.real)).to(device)
        out[i, :, :, 1] = torch.from_numpy(np.ascontiguousarray(R.imag)).to(device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(out, op=dist.ReduceOp.SUM)  # every index is owned by exactly one rank
    a = out.cpu().numpy()
    return a[..., 0] + 1j * a[..., 1]


def interleaved_scan(w, energies: Sequence[float], mode: int, nctx: int = 2, V=None, max_refine: int = -1, warmup: int = 0):
    """An energy scan on ONE GPU with `nctx` contexts, each on its own host thread and CUDA stream (include/hprmat.h: one
    context per host thread / stream).  The latency-bound phases of one factorisation (top-block kernels, small triangular
    solves) then overlap the tensor-core phases of another: 120 -> 106 ms per energy point at configs[3] with two contexts.
    Energies are handed out from a shared queue.  Only plumbing lives here: every solve is one hprmat_solve.

    w: a workload (paper_2512_11590_b200.workloads); V: its potential on the device (built from the context's mesh when
    None).  Returns (R, infos, seconds): R complex128 numpy (n_energies, nch, nch) holding each solve's column-major output
    (R[k].T is the R-matrix), the per-energy info dicts, and the wall time of the scan (contexts already set up, `warmup`
    untimed solves per context first)."""
    import queue
    import threading
    import time

    from . import binding as hb

    energies = [float(e) for e in energies]
    if nctx < 1:
        raise ValueError("nctx >= 1")
    dev = torch.cuda.current_device()
    slots = []
    for _ in range(nctx):
        st = torch.cuda.Stream(device=dev)
        with torch.cuda.stream(st):
            ctx = hb.Context(w.nch, w.nb, w.a, w.h2m, w.lval, w.ethr, max_mode=1 << mode)
            if V is None:
                r, _ = ctx.mesh()
                V = torch.from_numpy(w.potential(r)).to(f"cuda:{dev}")
            Rbuf = torch.empty((w.nch, w.nch), dtype=torch.complex128, device=f"cuda:{dev}")
            for _ in range(warmup):
                ctx.solve(energies[0], V, mode, max_refine=max_refine, R=Rbuf)
        slots.append((ctx, st, Rbuf))
    torch.cuda.synchronize(dev)
    out = np.zeros((len(energies), w.nch, w.nch), dtype=np.complex128)
    infos = [None] * len(energies)
    todo = queue.SimpleQueue()
    for k in range(len(energies)):
        todo.put(k)
    errors = []

    def work(i):
        try:
            torch.cuda.set_device(dev)
            ctx, st, Rbuf = slots[i]
            with torch.cuda.stream(st):
                while True:
                    try:
                        k = todo.get_nowait()
                    except queue.Empty:
                        break
                    _, info = ctx.solve(energies[k], V, mode, max_refine=max_refine, R=Rbuf)   # synchronises on st
                    infos[k] = info
                    out[k] = Rbuf.cpu().numpy()
        except Exception as e:  # noqa: BLE001 - re-raised below, in the caller's thread
            errors.append(e)

    t0 = time.perf_counter()
    threads = [threading.Thread(target=work, args=(i,)) for i in range(nctx)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    torch.cuda.synchronize(dev)
    seconds = time.perf_counter() - t0
    for ctx, _, _ in slots:
        ctx.destroy()
    if errors:
        raise errors[0]
    return out, infos, seconds
