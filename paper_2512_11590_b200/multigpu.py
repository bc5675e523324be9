"""Single LU factorisation distributed over several GPUs: partition, schedule and communication order.

The paper's multi-GPU solver (Type 6) distributes ONE N x N system over the GPUs of a node in cusolverMg's
1-D block-cyclic COLUMN layout and keeps the FP64 residual of the refinement on the host, which is what limits its gain
(53.1 -> 42.9 s on 1 -> 4 GPUs at N = 51200).  The design here:

  * columns in blocks of `nb` (1024 = the library's solve block), block k owned by rank k mod P; every rank holds its
    column blocks contiguously (local block index k // P), all N rows of them;
  * right-looking block step k:  the owner factors its N-k*nb by nb panel with partial pivoting (the library's recursive
    getrf on that column block) and BROADCASTS the factored panel (L11\\U11 on top, L21 below: <= 16 N nb bytes) together
    with the panel's row interchanges; every rank applies the interchanges to its own column blocks (left ones too, as
    LAPACK does), solves U12 = L11^-1 A12 on its blocks to the right and updates A22 -= L21 U12 there -- the tensor-core
    GEMM, all local.  One broadcast per block step is the only data-path collective (NCCL broadcast over NVLink/NVSwitch);
  * look-ahead: the owner of block k+1 updates that block first and factors it while the others still update -- expressed
    here by `schedule()` yielding the panel of k+1 before the trailing update of step k on the other blocks;
  * the right-hand sides (N x Nc) are replicated; forward/backward substitution walks the column blocks in order, each
    owner applying its block and broadcasting the updated right-hand-side slice (N/nb small broadcasts of nb x Nc);
  * the FP64 residual of the refinement is formed ON THE DEVICES from the structured operator (every rank has V and the
    tables: it is matrix-free), which removes the paper's host bottleneck.

This module holds the bookkeeping only -- ownership, local indices, the order of operations and of broadcasts -- and drives
an `ops` object that does the arithmetic: on a GPU node that is the library's kernels on each rank's column blocks; the
world_size-2 gloo test (tests/test_multigpu_gloo.py) passes a CPU stand-in to check the bookkeeping against a single-process
factorisation.  No timing claim is attached: this container has one GPU per run.
"""
from dataclasses import dataclass


@dataclass(frozen=True)
class BlockCyclic1D:
    """1-D block-cyclic distribution of the columns of an n x n matrix over `world` ranks."""
    n: int
    nb: int
    world: int

    @property
    def nblocks(self) -> int:
        return (self.n + self.nb - 1) // self.nb

    def owner(self, k: int) -> int:
        return k % self.world

    def local_index(self, k: int) -> int:
        return k // self.world

    def block_cols(self, k: int) -> range:
        return range(k * self.nb, min(self.n, (k + 1) * self.nb))

    def owned_blocks(self, rank: int) -> list:
        return [k for k in range(self.nblocks) if self.owner(k) == rank]

    def local_cols(self, rank: int) -> list:
        """global column indices held by `rank`, in local storage order"""
        return [j for k in self.owned_blocks(rank) for j in self.block_cols(k)]

    def local_offset(self, k: int) -> int:
        """first local column of block k on its owner"""
        return sum(len(self.block_cols(q)) for q in range(self.owner(k), k, self.world))

    def panel_bytes(self, k: int, elem_bytes: int = 16) -> int:
        """payload of block step k's broadcast: the factored panel (rows k*nb .. n) + its interchanges"""
        rows = self.n - k * self.nb
        return rows * len(self.block_cols(k)) * elem_bytes + 4 * len(self.block_cols(k))


def schedule(dist: BlockCyclic1D, lookahead: bool = True):
    """Order of operations of the right-looking factorisation as seen by EVERY rank (all ranks walk the same list):
         ("panel", k)            owner(k) factors block k's panel
         ("bcast", k)            owner(k) broadcasts panel k + interchanges
         ("swap",  k, blocks)    interchanges of panel k on these local blocks
         ("update", k, blocks)   U12 solve + A22 update of step k on these blocks (all > k)
    With look-ahead, block k+1 is updated and its panel factored before the rest of step k's update."""
    nblk = dist.nblocks
    for k in range(nblk):
        if not lookahead or k == 0:
            yield ("panel", k)
        yield ("bcast", k)
        others = [q for q in range(nblk) if q != k]
        yield ("swap", k, others)
        right = [q for q in range(k + 1, nblk)]
        if lookahead and k + 1 < nblk:
            yield ("update", k, [k + 1])
            yield ("panel", k + 1)
            right = right[1:]
        if right:
            yield ("update", k, right)


def factor(dist: BlockCyclic1D, rank: int, local, ops, broadcast, lookahead: bool = True):
    """Run the schedule on this rank.  `local`: this rank's column blocks (an ops-defined container holding all n rows of
    its columns).  ops provides
         ops.panel(local, off, k0, w) -> (panel, piv)    factor rows k0.. of local columns off..off+w in place
         ops.swap(local, off, w, k0, piv)                apply the interchanges of a panel starting at row k0
         ops.update(local, off, w, k0, kw, panel)        U12 = L11^-1 A12 and A22 -= L21 U12 on local columns off..off+w
    broadcast(obj, src) -> obj is the collective (torch.distributed broadcast of the panel buffer on a GPU node).
    Returns the list of (k, pivots) in factorisation order."""
    mine = set(dist.owned_blocks(rank))
    panels = {}     # panels factored locally, waiting for their broadcast
    received = {}
    pivots = []
    for step in schedule(dist, lookahead):
        kind, k = step[0], step[1]
        k0, kw = k * dist.nb, len(dist.block_cols(k))
        if kind == "panel":
            if k in mine:
                panels[k] = ops.panel(local, dist.local_offset(k), k0, kw)
        elif kind == "bcast":
            received[k] = broadcast(panels.pop(k) if k in mine else None, dist.owner(k))
            pivots.append((k, received[k][1]))
        elif kind == "swap":
            for q in step[2]:
                if q in mine:
                    ops.swap(local, dist.local_offset(q), len(dist.block_cols(q)), k0, received[k][1])
        elif kind == "update":
            for q in step[2]:
                if q in mine:
                    ops.update(local, dist.local_offset(q), len(dist.block_cols(q)), k0, kw, received[k][0])
    return pivots
