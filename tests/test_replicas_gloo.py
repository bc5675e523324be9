"""The N > 1 path (replicas over an energy scan) on CPU: world_size 2, gloo, 127.0.0.1.  Covers the
rank -> energy assignment, the gather of the R-matrices in scan order and the max-over-ranks timing rule.  The per-rank
'solve' here is a stand-in that depends on the scan index only -- the point is the bookkeeping, not the arithmetic."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2512_11590_b200 import scan


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _fake_R(i, nch):
    k = np.arange(nch)
    return (i + 1) * (np.add.outer(k, 2 * k) + 1j * np.subtract.outer(k, k + i))


def _worker(rank, world, port, n_energies, nch, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = scan.shard_indices(n_energies, rank, world)
        local = {i: _fake_R(i, nch) for i in mine}
        allR = scan.gather_rmatrices(local, n_energies, nch)
        tmax = scan.max_over_ranks(1.0 + rank)
        q.put((rank, mine, allR, tmax))
    finally:
        dist.destroy_process_group()


def test_scan_replicas_world2_gloo():
    world, n_energies, nch = 2, 5, 3
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_energies, nch, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    seen = []
    for rank, mine, allR, tmax in got:
        assert mine == list(range(rank, n_energies, world))
        seen += mine
        assert tmax == 2.0                                    # the slowest rank's time, on every rank
        for i in range(n_energies):
            assert np.array_equal(allR[i], _fake_R(i, nch))   # scan order, every rank holds all of them
    assert sorted(seen) == list(range(n_energies))            # a partition: nothing dropped, nothing twice


def test_shard_and_bench_energy_rules():
    assert scan.shard_indices(10, 0, 4) == [0, 4, 8] and scan.shard_indices(10, 3, 4) == [3, 7]
    assert scan.shard_indices(2, 3, 4) == []
    e = [5.0, 10.0, 15.0]
    assert [scan.bench_energy(e, r) for r in range(5)] == [5.0, 10.0, 15.0, 20.0, 25.0]
    assert [scan.bench_energy([30.0], r) for r in range(3)] == [30.0, 30.5, 31.0]
    assert scan.max_over_ranks(3.5) == 3.5                   # no process group: identity
    R = scan.gather_rmatrices({0: np.eye(2)}, 1, 2)
    assert R.shape == (1, 2, 2) and np.array_equal(R[0], np.eye(2))
