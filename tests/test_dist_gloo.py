"""Host logic of the N > 1 launch (paper_2302_09708_b200/dist.py) on CPU: the paper's column / row partition
 and the max-over-ranks reduction, with two gloo processes."""
import os
import socket

import numpy as np
import pytest

from paper_2302_09708_b200 import dist as pdist


def test_partition_matches_paper_rule():
    # equal sizes on all ranks but the last, which gets the remainder
    for n in (0, 1, 7, 32, 256, 7680, 1327104):
        for p in (1, 2, 3, 4, 8):
            parts = pdist.partition_all(n, p)
            assert parts[0][0] == 0 and parts[-1][1] == n
            sizes = [e - b for b, e in parts]
            assert sum(sizes) == n
            for k in range(p - 1):
                assert parts[k][1] == parts[k + 1][0]
            full = [s for s in sizes if s == sizes[0]]
            assert all(s <= sizes[0] for s in sizes)
            if n >= p and n % p == 0:
                assert len(full) == p
    assert pdist.partition(10, 4, 3) == (9, 10)
    assert pdist.partition(10, 4, 0) == (0, 3)
    with pytest.raises(ValueError):
        pdist.partition(10, 0, 0)


def test_column_blocks_cover_range():
    blocks = pdist.column_blocks(3840, 7680, 1024)
    assert blocks[0] == (3840, 4864) and blocks[-1] == (6912, 7680)
    assert sum(e - b for b, e in blocks) == 3840


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # each rank "filters" its column slice of a shared synthetic block: disjoint slices that tile the block
        ns = 37
        b, e = pdist.partition(ns, world, rank)
        mine = torch.zeros(ns, dtype=torch.float64)
        mine[b:e] = 1.0
        dist.all_reduce(mine)
        covered = bool(torch.equal(mine, torch.ones(ns, dtype=torch.float64)))
        times = pdist.max_over_ranks([1.0 + rank, 5.0 - rank])
        units = pdist.sum_over_ranks([float(e - b)])
        pdist.barrier()
        out.put((rank, covered, times, units))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_reduction():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, covered, times, units in res:
        assert covered
        assert times == [2.0, 5.0]           # max over ranks of [1, 5] and [2, 4]
        assert units == [37.0]
    assert np.isfinite(res[0][2]).all()
