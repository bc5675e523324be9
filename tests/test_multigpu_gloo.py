"""Bookkeeping of the distributed single LU (paper_2512_11590_b200/multigpu.py) with
world_size 2 on gloo and a CPU STAND-IN for the kernels: ownership, local offsets, broadcast order and look-ahead must
reproduce a single-process LU with partial pivoting.  CPU only; the stand-in arithmetic (numpy) lives here, not in the
product."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2512_11590_b200.multigpu import BlockCyclic1D, factor, schedule


class NumpyOps:
    """unblocked partial-pivoting panel, row swaps, triangular solve + update -- the stand-in for the CUDA kernels"""

    @staticmethod
    def panel(local, off, k0, w):
        P = local[k0:, off:off + w]
        piv = np.zeros(w, dtype=np.int64)
        for j in range(min(w, P.shape[0])):
            p = j + int(np.argmax(np.abs(P[j:, j].real) + np.abs(P[j:, j].imag)))
            piv[j] = p
            if p != j:
                P[[j, p], :] = P[[p, j], :]
            P[j + 1:, j] /= P[j, j]
            P[j + 1:, j + 1:] -= np.outer(P[j + 1:, j], P[j, j + 1:])
        return P.copy(), piv

    @staticmethod
    def swap(local, off, w, k0, piv):
        blk = local[k0:, off:off + w]
        for j, p in enumerate(piv):
            if p != j:
                blk[[j, p], :] = blk[[p, j], :]

    @staticmethod
    def update(local, off, w, k0, kw, panel):
        L11 = np.tril(panel[:kw, :kw], -1) + np.eye(kw)
        A12 = local[k0:k0 + kw, off:off + w]
        A12[:] = np.linalg.solve(L11, A12)
        local[k0 + kw:, off:off + w] -= panel[kw:, :kw] @ A12


def test_block_cyclic_maps():
    d = BlockCyclic1D(n=10, nb=3, world=2)
    assert d.nblocks == 4 and [d.owner(k) for k in range(4)] == [0, 1, 0, 1]
    assert d.local_cols(0) == [0, 1, 2, 6, 7, 8] and d.local_cols(1) == [3, 4, 5, 9]
    assert [d.local_offset(k) for k in range(4)] == [0, 0, 3, 3]
    assert d.panel_bytes(1) == (10 - 3) * 3 * 16 + 12
    steps = list(schedule(d))
    # every panel is factored exactly once, before its broadcast; with look-ahead panel k+1 precedes the rest of update k
    for k in range(4):
        assert steps.index(("panel", k)) < steps.index(("bcast", k))
        assert sum(1 for s in steps if s[:2] == ("panel", k)) == 1
    assert steps.index(("panel", 1)) < steps.index(("update", 0, [2, 3]))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n, nb, lookahead, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rng = np.random.default_rng(7)
        A = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))       # same matrix on every rank (seeded)
        d = BlockCyclic1D(n=n, nb=nb, world=world)
        local = np.asfortranarray(A[:, d.local_cols(rank)])
        order = []

        def bcast(obj, src):
            order.append(src)
            box = [obj]
            dist.broadcast_object_list(box, src=src)
            return box[0]

        piv = factor(d, rank, local, NumpyOps, bcast, lookahead=lookahead)
        gathered = [None] * world
        dist.all_gather_object(gathered, (d.local_cols(rank), local))
        if rank == 0:
            LU = np.zeros((n, n), dtype=complex)
            for cols, blk in gathered:
                LU[:, cols] = blk
            perm = np.arange(n)
            for k, pv in piv:
                for j, p in enumerate(pv):
                    a, b = k * nb + j, k * nb + int(p)
                    perm[[a, b]] = perm[[b, a]]
            L = np.tril(LU, -1) + np.eye(n)
            U = np.triu(LU)
            out["err"] = float(np.abs(L @ U - A[perm]).max() / np.abs(A).max())
            out["maxL"] = float(np.abs(np.tril(LU, -1)).max())
            out["order"] = order
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n,nb,lookahead", [(37, 8, True), (37, 8, False), (64, 16, True), (50, 7, True)])
def test_distributed_lu_matches_single_process(n, nb, lookahead):
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), n, nb, lookahead, out), nprocs=world, join=True)
    assert out["err"] < 1e-12, dict(out)
    assert out["maxL"] <= 2.0 ** 0.5 + 1e-12     # partial pivoting on |re| + |im| (the library's rule): |l| <= sqrt(2)
    nblk = (n + nb - 1) // nb
    assert list(out["order"]) == [k % world for k in range(nblk)]   # one broadcast per block step, from its owner, in order
