"""Multi-GPU data path of one CheFSI step, one process per GPU over
torch.distributed: plumbing only -- every arithmetic step runs in the kernels behind the C ABI (a `local` operator object).

The paper distributes the step two ways (eqs. (1)-(2)): a column-wise partition
X = [X_(1) ... X_(p)] for the filter (no communication, eq. (4), 190) and a row-wise
partition X = [X^(1); ...; X^(p)] for projection / rotation, with a redistribution in between
(eq. (5), 168-170).  "If N_d and N_s are not integer multiples of the number of processors, the number of
rows and columns for the p-th processor are reduced, such that the sizes of the matrices are the same on the remaining
processors": every rank but the last owns ceil(n/p) items, the last one what is left.

    filter     column partition, rank k filters its columns X_(k) and forms Y_(k) = H X_(k)
    a2a        X_(k), Y_(k) -> row blocks X~^(k), Y~^(k): ONE all-to-all each, GPU-direct (NCCL over NVLink / NVSwitch);
               the paper stages both through the host and MPI
    project    H~^(k) = X~^(k)T Y~^(k), M~^(k) = X~^(k)T X~^(k) locally, then all-reduce(sum) of the two N_s x N_s
               matrices (eqs. 6-8; NVSwitch reduces in the switch when NCCL enables NVLS)
    solve      every rank solves the N_s x N_s eigenproblem redundantly on its own GPU (the paper: root rank + broadcast,
               PAPER.md:150-158), or takes Q from the caller
    rotate     X^(k) = X~^(k) Z~ on the local rows (eqs. 10-11)
    a2a back   row blocks -> column partition for the next filter

Layout.  A local block of r rows x c columns (column-major, ld = r) is a (c, r) tensor contiguous along its last axis.
The send buffer of the column->row all-to-all is the list over destination ranks d of the (c_me, rows_d) slices; what rank d
receives from all sources, concatenated in rank order, IS the (N_s, rows_d) tensor of its row block: no unpacking.  The way
back is the mirror image.

`local` supplies the kernels: filter(X, ...), apply(X) -> Y, gram(A, B, nrows, symmetric) -> (n, m) tensor,
rotate_rows(X, nrows, Q), eigensolve(Hs, Ms) -> (D, Z).  On a GPU that is `SparcGpuLocal` below (the C ABI); the CPU gloo
tests pass an oracle-backed stand-in so that the partition / redistribution / reduction logic runs with world_size 2.
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple


def partition(n: int, p: int, k: int) -> Tuple[int, int]:
    """[begin, end) of the items (columns for eq. (1), rows for eq. (2)) that rank k of p owns."""
    if p < 1 or not (0 <= k < p) or n < 0:
        raise ValueError("partition: need p >= 1, 0 <= k < p, n >= 0")
    size = -(-n // p)                      # ceil(n / p): equal on all ranks but the last
    begin = min(k * size, n)
    end = min(begin + size, n)
    return begin, end


def partition_all(n: int, p: int) -> List[Tuple[int, int]]:
    return [partition(n, p, k) for k in range(p)]


def column_blocks(begin: int, end: int, col_block: int) -> List[Tuple[int, int]]:
    """Column blocks [j0, j1) that one rank filters one after the other."""
    if col_block <= 0:
        raise ValueError("col_block must be positive")
    return [(j, min(j + col_block, end)) for j in range(begin, end, col_block)]


def _world():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        return dist.get_world_size(), dist.get_rank()
    return 1, 0


def max_over_ranks(values: Sequence[float], device=None) -> List[float]:
    """Element-wise MAX over all ranks of a short list of timings (identity without a process group)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if _world()[0] > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def sum_over_ranks(values: Sequence[float], device=None) -> List[float]:
    """Element-wise SUM over all ranks (work units processed by the whole job)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if _world()[0] > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.cpu()]


def barrier(device=None) -> None:
    """Process-group barrier (if any) followed by a device synchronize (if a CUDA device is given)."""
    import torch
    import torch.distributed as dist
    if _world()[0] > 1:
        dist.barrier()
    if device is not None and torch.cuda.is_available():
        torch.cuda.synchronize(device)


# ----------------------------------------------------------------------------------------------------------------------
# redistribution between the two partitions, by column blocks (temporaries stay block-sized: at config 4 the orbitals are
# 81.5 GB, so a rank can afford its column slice, its row slice and nothing else of that size)
# ----------------------------------------------------------------------------------------------------------------------
FORCE_COLLECTIVES = False      # tests: issue the collectives even in a one-rank group (exercises NCCL on a single GPU)


def _a2a(recv, send, out_splits, in_splits, async_op: bool = False):
    """all-to-all of flat buffers.  async_op: returns the collective's work handle (None when no collective was issued);
    the caller keeps `send` / `recv` alive and calls .wait() before it touches `recv`."""
    import torch.distributed as dist
    if _world()[0] == 1 and not (FORCE_COLLECTIVES and dist.is_initialized()):
        recv.copy_(send)
        return None
    return dist.all_to_all_single(recv, send, output_split_sizes=out_splits, input_split_sizes=in_splits, async_op=async_op)


def _block_counts(ns: int, p: int, j0: int, j1: int) -> List[int]:
    """How many of its local columns [j0, j1) each rank actually owns (the last rank may own fewer, or none)."""
    out = []
    for cb, ce in partition_all(ns, p):
        c = ce - cb
        out.append(max(0, min(j1, c) - min(j0, c)))
    return out


def block_columns_to_rows(Xb, nd: int, ns: int, j0: int, j1: int, async_op: bool = False):
    """Xb: (nb_me, ld >= nd) = this rank's local columns [j0, j1) (clipped to what it owns).  Returns the (sum_s nb_s, r_me)
    tensor of this rank's rows of the same local column range of EVERY rank, grouped by source rank, and
    the per-rank column counts.  async_op: the all-to-all is only started; a third value (work handle or None, send buffer)
    is returned and the caller waits on the handle before reading the tensor."""
    import torch
    p, me = _world()
    rows = partition_all(nd, p)
    r_me = rows[me][1] - rows[me][0]
    nbs = _block_counts(ns, p, j0, j1)
    nb_me = nbs[me]
    assert Xb.shape[0] == nb_me
    send = torch.cat([Xb[:, b:e].reshape(-1) for b, e in rows]) if nb_me > 0 else Xb.new_empty(0)
    recv = Xb.new_empty(sum(nbs) * r_me)
    work = _a2a(recv, send, [n * r_me for n in nbs], [nb_me * (e - b) for b, e in rows], async_op=async_op)
    if async_op:
        return recv.view(sum(nbs), r_me), nbs, (work, send)
    return recv.view(sum(nbs), r_me), nbs


def block_rows_to_columns(Xr, nd: int, ns: int, j0: int, j1: int, out):
    """Inverse of block_columns_to_rows for the local column range [j0, j1): Xr is the whole (ns, r_me) row block of this
    rank; `out` (nb_me, ld >= nd) receives this rank's columns [j0, j1)."""
    import torch
    p, me = _world()
    rows = partition_all(nd, p)
    cols = partition_all(ns, p)
    r_me = rows[me][1] - rows[me][0]
    nbs = _block_counts(ns, p, j0, j1)
    nb_me = nbs[me]
    assert out.shape[0] == nb_me
    parts = [Xr[cols[s][0] + j0: cols[s][0] + j0 + nbs[s]].reshape(-1) for s in range(p)]
    send = torch.cat(parts)
    recv = Xr.new_empty(nb_me * nd)
    _a2a(recv, send, [nb_me * (e - b) for b, e in rows], [n * r_me for n in nbs])
    off = 0
    for b, e in rows:                          # the piece from rank s holds rows [b, e) of my columns
        if nb_me > 0:
            out[:, b:e].copy_(recv[off:off + nb_me * (e - b)].view(nb_me, e - b))
        off += nb_me * (e - b)
    return out


def columns_to_rows(Xc, nd: int, ns: int, col_block: int = 0):
    """Column partition -> row partition of a whole block.  Xc: (c_me, ld >= nd).  Returns the (ns, r_me) tensor of this
    rank's rows [partition(nd, p, k))."""
    p, me = _world()
    rows = partition_all(nd, p)
    cols = partition_all(ns, p)
    c_me = cols[me][1] - cols[me][0]
    r_me = rows[me][1] - rows[me][0]
    assert Xc.shape[0] == c_me and Xc.shape[1] >= nd
    c_max = cols[0][1] - cols[0][0]
    cbk = col_block if col_block > 0 else 1024
    Xr = Xc.new_empty((ns, r_me))
    for j0 in range(0, c_max, cbk):            # the same number of collectives on every rank
        j1 = min(j0 + cbk, c_max)
        blk, nbs = block_columns_to_rows(Xc[min(j0, c_me):min(j1, c_me)], nd, ns, j0, j1)
        off = 0
        for s in range(p):
            Xr[cols[s][0] + j0: cols[s][0] + j0 + nbs[s]].copy_(blk[off:off + nbs[s]])
            off += nbs[s]
    return Xr


def rows_to_columns(Xr, nd: int, ns: int, out=None, col_block: int = 0):
    """Row partition -> column partition of a whole block.  Xr: (ns, r_me).  Returns (or fills `out`, (c_me, ld >= nd))."""
    p, me = _world()
    rows = partition_all(nd, p)
    cols = partition_all(ns, p)
    c_me = cols[me][1] - cols[me][0]
    r_me = rows[me][1] - rows[me][0]
    assert tuple(Xr.shape) == (ns, r_me)
    if out is None:
        out = Xr.new_empty((c_me, nd))
    c_max = cols[0][1] - cols[0][0]
    cbk = col_block if col_block > 0 else 1024
    for j0 in range(0, c_max, cbk):
        j1 = min(j0 + cbk, c_max)
        block_rows_to_columns(Xr, nd, ns, j0, j1, out[min(j0, c_me):min(j1, c_me)])
    return out


# ----------------------------------------------------------------------------------------------------------------------
# the distributed step
# ----------------------------------------------------------------------------------------------------------------------
class SparcGpuLocal:
    """The local kernels of the distributed step: thin adapter over api.SparcGpu (C ABI, this rank's GPU)."""

    def __init__(self, g):
        self.g = g

    def filter(self, X, degree, a, b, a0, col_block=0):
        return self.g.chebyshev_filter(X, degree, a, b, a0, col_block=col_block)

    def apply(self, X):
        return self.g.hamiltonian_apply(X)

    def gram(self, A, B, nrows, symmetric):
        return self.g.gram(A, B, nrows, symmetric=symmetric)

    def rotate_rows(self, X, nrows, Q):
        return self.g.rotate_rows(X, nrows, Q)

    def eigensolve(self, Hs, Ms):
        D, Z, _ = self.g.eigensolve(Hs, Ms)
        return D, Z


def chefsi_step(local, Xc, nd: int, ns: int, degree: int, a: float, b: float, a0: float, Q=None, col_block: int = 0,
                timers: Optional[dict] = None):
    """One distributed CheFSI step.  Xc: this rank's columns (c_me, ld >= nd) of Psi, overwritten with its columns of the
    rotated block.  Q: (ns, ns) tensor holding the column-major rotation, or None to solve Hs Z = Ms Z D on the device.
    Returns (Hs, Ms, D or None): the reduced subspace matrices ((ns, ns) tensors holding the column-major matrices),
    identical on every rank.  `timers`: optional {'mark': fn(name)}, called between the phases (bench.py records events)."""
    import torch.distributed as dist
    p, me = _world()
    mark = (timers or {}).get("mark", lambda name: None)
    rows = partition_all(nd, p)
    cols = partition_all(ns, p)
    r_me = rows[me][1] - rows[me][0]
    c_me = cols[me][1] - cols[me][0]
    c_max = cols[0][1] - cols[0][0]
    cbk = col_block if col_block > 0 else 1024
    mark("start")
    # Filter and redistribution, pipelined by column blocks (columns are independent in the filter): the
    # all-to-all of block j is started asynchronously (it runs on the process group's own stream) and the filter of block
    # j + 1 is queued behind it on the compute stream, so the NVLink transfer of one block hides under the kernels of the
    # next.  At most two blocks' send / receive buffers are alive at a time.  The filter's result does not depend on how
    # its columns are blocked (R19), so this equals filtering the whole slice first.
    Xr = Xc.new_empty((ns, r_me))

    def finish(item):
        j0, blk, nbs, (work, _send) = item
        if work is not None:
            work.wait()
        off = 0
        for s in range(p):
            Xr[cols[s][0] + j0: cols[s][0] + j0 + nbs[s]].copy_(blk[off:off + nbs[s]])
            off += nbs[s]

    pending = None
    for j0 in range(0, c_max, cbk):            # the same number of collectives on every rank
        j1 = min(j0 + cbk, c_max)
        Xb = Xc[min(j0, c_me):min(j1, c_me)]
        if Xb.shape[0] > 0:
            local.filter(Xb, degree, a, b, a0, col_block)
        cur = (j0,) + block_columns_to_rows(Xb, nd, ns, j0, j1, async_op=True)
        if pending is not None:
            finish(pending)
        pending = cur
    if pending is not None:
        finish(pending)
    mark("filter")                             # filter and redistribution overlap: "to_rows" is what is left exposed
    mark("to_rows")
    # H~ = sum_k X~^(k)T Y~^(k) by column blocks of Y = H X: a block is formed in the column partition, redistributed and
    # contracted with the whole local row block; column j of Hs is row j of the (ns, ns) tensor
    Hs = Xr.new_zeros((ns, ns))
    for j0 in range(0, c_max, cbk):
        j1 = min(j0 + cbk, c_max)
        Xb = Xc[min(j0, c_me):min(j1, c_me)]
        Yb = local.apply(Xb) if Xb.shape[0] > 0 else Xb
        Yr, nbs = block_columns_to_rows(Yb, nd, ns, j0, j1)
        G = local.gram(Xr, Yr, r_me, False)             # (sum nbs, ns): the block's columns of this rank's partial Hs
        off = 0
        for s in range(p):
            Hs[cols[s][0] + j0: cols[s][0] + j0 + nbs[s]].copy_(G[off:off + nbs[s]])
            off += nbs[s]
        del Yb, Yr, G
    Ms = local.gram(Xr, Xr, r_me, True)
    if p > 1 or (FORCE_COLLECTIVES and dist.is_initialized()):
        dist.all_reduce(Hs)
        dist.all_reduce(Ms)
    mark("project")
    D = None
    if Q is None:
        D, Q = local.eigensolve(Hs, Ms)
    mark("solve")
    local.rotate_rows(Xr, r_me, Q)
    mark("rotate")
    rows_to_columns(Xr, nd, ns, out=Xc, col_block=cbk)
    mark("to_columns")
    return Hs, Ms, D
