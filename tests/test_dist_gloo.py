"""The N > 1 data path (paper_2302_09708_b200/dist.py) on CPU with two and with three gloo processes: the paper's column / row partitions
(PAPER.md:104-108), the column <-> row redistributions, the all-reduce of the partial subspace
matrices and the whole distributed step, with the local kernels replaced by the oracle (the CUDA kernels
need a GPU; tests may call oracle/) and the result compared with the single-process oracle."""
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


class OracleLocal:
    """Stand-in for the CUDA kernels in the CPU test: the same five local operations, computed by the oracle."""

    def __init__(self, wl):
        from oracle import oracle as orc
        self.orc = orc
        self.H = orc.Hamiltonian(wl)
        self.nd = wl.nd

    def _np(self, X, rows):
        return np.asfortranarray(X[:, :rows].numpy().T)

    def filter(self, X, degree, a, b, a0, col_block=0):
        import torch
        F = self.H.chebyshev_filter(self._np(X, self.nd), degree, a, b, a0)
        X[:, :self.nd] = torch.from_numpy(np.ascontiguousarray(F.T))
        return X

    def apply(self, X):
        import torch
        Y = torch.zeros_like(X)
        Y[:, :self.nd] = torch.from_numpy(np.ascontiguousarray(self.H.apply(self._np(X, self.nd)).T))
        return Y

    def gram(self, A, B, nrows, symmetric):
        import torch
        G = self.orc.gram(self._np(A, nrows), self._np(B, nrows)) if nrows > 0 else np.zeros((A.shape[0], B.shape[0]))
        return torch.from_numpy(np.ascontiguousarray(G.T))

    def rotate_rows(self, X, nrows, Q):
        import torch
        if nrows > 0:
            R = self.orc.rotate(self._np(X, nrows), np.asfortranarray(Q.numpy().T))
            X[:, :nrows] = torch.from_numpy(np.ascontiguousarray(R.T))
        return X

    def eigensolve(self, Hs, Ms):
        import torch
        D, Z = self.orc.sygv(np.asfortranarray(Hs.numpy().T), np.asfortranarray(Ms.numpy().T))
        return torch.from_numpy(D), torch.from_numpy(np.ascontiguousarray(Z.T))


def _make_wl():
    from paper_2302_09708_b200 import workloads as wlmod
    pos = np.array([[1.0, 2.0, 3.0], [4.5, 5.0, 0.4]])
    return wlmod.make_custom("dist", (13, 15, 15), (0.5, 0.45, 0.4), (0, 0, 1), 7, 4, pos, [4, 9], 2.3, seed=51)


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # reductions used by bench.py
        times = pdist.max_over_ranks([1.0 + rank, 5.0 - rank])
        units = pdist.sum_over_ranks([3.0 + rank])
        # redistribution round trip on a labelled block: element (i, j) = i + 10000 j
        nd, ns = 37, 5                       # world 3: rows 13 + 13 + 11, columns 2 + 2 + 1
        cb, ce = pdist.partition(ns, world, rank)
        rb, re_ = pdist.partition(nd, world, rank)
        full = (np.arange(nd)[:, None] + 10000.0 * np.arange(ns)[None, :])
        Xc = torch.zeros((ce - cb, nd + 3), dtype=torch.float64)
        Xc[:, :nd] = torch.from_numpy(np.ascontiguousarray(full[:, cb:ce].T))
        Xr = pdist.columns_to_rows(Xc, nd, ns, col_block=2)      # blocks with a ragged tail: the ranks own 3 and 2 columns
        rows_ok = bool(np.array_equal(Xr.numpy().T, full[rb:re_, :]))
        back = torch.zeros_like(Xc)
        pdist.rows_to_columns(Xr, nd, ns, out=back, col_block=2)
        round_ok = bool(torch.equal(back, Xc))
        # the whole step, caller's Q and device-side solve
        wl = _make_wl()
        local = OracleLocal(wl)
        cb, ce = pdist.partition(wl.ns, world, rank)
        X = wl.psi_columns(range(wl.ns))
        rng = np.random.default_rng(5)
        Q = np.linalg.qr(rng.standard_normal((wl.ns, wl.ns)))[0]
        res = {}
        for mode in ("given_q", "solve"):
            Xc = torch.from_numpy(np.ascontiguousarray(X[:, cb:ce].T)).clone()
            Qt = torch.from_numpy(np.ascontiguousarray(Q.T)) if mode == "given_q" else None
            Hs, Ms, D = pdist.chefsi_step(local, Xc, wl.nd, wl.ns, wl.degree, wl.a, wl.b, wl.a0, Q=Qt,
                                            col_block=0 if mode == "given_q" else 3)
            res[mode] = (Xc.numpy().T.copy(), Hs.numpy().T.copy(), Ms.numpy().T.copy(), None if D is None else D.numpy().copy())
        pdist.barrier()
        out.put((rank, times, units, rows_ok, round_ok, (cb, ce), res))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_gloo_step_matches_single_process_oracle(world):
    """world 2: 7 orbitals as 4 + 3; world 3: 3 + 3 + 1 (ragged last rank), 37 labelled rows as 13 + 13 + 11."""
    import torch.multiprocessing as mp
    from oracle import oracle as orc
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, times, units, rows_ok, round_ok, _, _ in res:
        assert times == [float(world), 5.0]   # max over ranks of [1 + rank, 5 - rank]
        assert units == [3.0 * world + world * (world - 1) / 2]
        assert rows_ok and round_ok
    # single-process reference: filter -> project -> (Q | solve) -> rotate
    wl = _make_wl()
    H = orc.Hamiltonian(wl)
    X = wl.psi_columns(range(wl.ns))
    F = H.chebyshev_filter(X, wl.degree, wl.a, wl.b, wl.a0)
    Hs_o, Ms_o = H.project(F)
    rng = np.random.default_rng(5)
    Q = np.linalg.qr(rng.standard_normal((wl.ns, wl.ns)))[0]
    R_given = orc.rotate(F, Q)
    D_o, Z_o = orc.sygv(0.5 * (Hs_o + Hs_o.T), Ms_o)
    for mode in ("given_q", "solve"):
        got = np.concatenate([r[6][mode][0] for r in res], axis=1)        # columns of rank 0, then rank 1
        for r in res:
            Hs, Ms = r[6][mode][1], r[6][mode][2]
            assert np.linalg.norm(Hs - Hs_o) <= 1e-12 * np.linalg.norm(Hs_o)
            assert np.linalg.norm(Ms - Ms_o) <= 1e-12 * np.linalg.norm(Ms_o)
        for r in res[1:]:                                                # the all-reduced matrices are the same on every rank
            assert np.array_equal(res[0][6][mode][1], r[6][mode][1])
        if mode == "given_q":
            assert np.linalg.norm(got - R_given) <= 1e-12 * np.linalg.norm(R_given)
        else:
            D = res[0][6][mode][3]
            assert np.max(np.abs(D - D_o)) <= 1e-10 * max(1.0, np.abs(D_o).max())
            # rotated block: M-orthonormal Ritz vectors with Rayleigh quotients D
            Hs2, Ms2 = H.project(got)
            assert np.max(np.abs(Ms2 - np.eye(wl.ns))) <= 1e-9
            assert np.max(np.abs(Hs2 - np.diag(D))) <= 1e-9 * max(1.0, np.abs(D).max())
