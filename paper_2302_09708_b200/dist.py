"""Host-side logic of the multi-process launch (no arithmetic of the method lives here).

The paper distributes the path two ways (eqs. (1)-(2)): a column-wise partition
X = [X_(1) ... X_(p)] for the filter (no communication, eq. (4), 190) and a row-wise
partition X = [X^(1); ...; X^(p)] for projection / rotation.  "If N_d and N_s are not integer multiples of
the number of processors, the number of rows and columns for the p-th processor are reduced, such that the
sizes of the matrices are the same on the remaining processors": every rank but the last
owns ceil(n/p) items, the last one owns what is left.

north_star fixes "everything runs on one GPU", so this build runs N independent replicas under torchrun
("replicas only"): the only cross-rank traffic is the barrier and the max-over-ranks
of the device timers, both here.  The partition helpers are what a real column/row distribution (SURVEY.md
section 8(e), listed as next) would start from; they are exercised by a world-size-2 gloo test.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple


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


def max_over_ranks(values: Sequence[float], device=None) -> List[float]:
    """Element-wise MAX over all ranks of a short list of timings (identity without a process group)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def sum_over_ranks(values: Sequence[float], device=None) -> List[float]:
    """Element-wise SUM over all ranks (work units processed by the whole job)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.cpu()]


def barrier(device=None) -> None:
    """Process-group barrier (if any) followed by a device synchronize (if a CUDA device is given)."""
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
    if device is not None and torch.cuda.is_available():
        torch.cuda.synchronize(device)
