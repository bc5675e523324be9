"""Energy-scan bookkeeping for N > 1 GPUs (replicas only).

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
