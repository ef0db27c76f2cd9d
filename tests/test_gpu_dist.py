"""The distributed CheFSI step (paper_2302_09708_b200/dist.py) with the real CUDA kernels
behind it, on ONE GPU: a one-rank NCCL group with the collectives forced on, so that the blocked column <-> row
redistribution, the all-reduce and the local kernels (sparc_gpu_gram, sparc_gpu_rotate_rows, sparc_gpu_eigensolve) run
exactly as they do with N ranks; the two-rank logic itself is covered on CPU by tests/test_dist_gloo.py.  Compared with the
single-process oracle at the gates of the real path."""
import os
import socket

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2302_09708_b200 import workloads as wlmod

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


@pytest.fixture(scope="module")
def api():
    from paper_2302_09708_b200 import api as a
    return a


@pytest.fixture(scope="module")
def nccl_group(torch):
    import torch.distributed as dist
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    yield dist
    dist.destroy_process_group()


def fro(G, O):
    return float(np.linalg.norm(G - O) / np.linalg.norm(O))


@pytest.mark.parametrize("forced", [False, True])
def test_distributed_step_one_rank(torch, api, nccl_group, forced):
    from paper_2302_09708_b200 import dist as pdist
    wl = wlmod.make_workload(0)
    g = api.SparcGpu(wl)
    local = pdist.SparcGpuLocal(g)
    H = orc.Hamiltonian(wl)
    X = wl.psi()
    F = H.chebyshev_filter(X, wl.degree, wl.a, wl.b, wl.a0)
    Hs_o, Ms_o = H.project(F)
    Q = wl.q_matrix()
    R_o = orc.rotate(F, Q)
    pdist.FORCE_COLLECTIVES = forced
    try:
        # caller's Q, several column blocks with a ragged tail
        Xc = api.colmajor_from_numpy(X, ld=wl.nd + 4)
        launches0 = g.get_info("kernel_launches")
        Hs, Ms, D = pdist.chefsi_step(local, Xc, wl.nd, wl.ns, wl.degree, wl.a, wl.b, wl.a0,
                                      Q=api.colmajor_from_numpy(Q), col_block=12)
        assert g.get_info("kernel_launches") > launches0 and D is None
        e = (fro(api.colmajor_to_numpy(Xc, wl.nd), R_o), fro(api.colmajor_to_numpy(Hs), Hs_o), fro(api.colmajor_to_numpy(Ms), Ms_o))
        print(f"[parity] distributed step (1 rank, collectives forced: {forced}): Psi Q {e[0]:.2e}, Hs {e[1]:.2e}, Ms {e[2]:.2e}")
        assert max(e) <= 1e-11 and max(e) <= 1e-13
        # device-side solve: M-orthonormal Ritz vectors with Rayleigh quotients D; D matches the oracle's sygv
        Xc = api.colmajor_from_numpy(X)
        Hs, Ms, D = pdist.chefsi_step(local, Xc, wl.nd, wl.ns, wl.degree, wl.a, wl.b, wl.a0, Q=None)
        Dn = D.cpu().numpy()
        Do, _ = orc.sygv(0.5 * (Hs_o + Hs_o.T), Ms_o)
        assert np.max(np.abs(Dn - Do)) <= 1e-11 * max(1.0, np.abs(Do).max())
        Hs2, Ms2 = g.project(Xc)
        assert np.max(np.abs(api.colmajor_to_numpy(Ms2) - np.eye(wl.ns))) <= 1e-9
        assert np.max(np.abs(api.colmajor_to_numpy(Hs2) - np.diag(Dn))) <= 1e-9 * max(1.0, np.abs(Dn).max())
    finally:
        pdist.FORCE_COLLECTIVES = False
        g.close()


def test_gram_and_rotate_rows_entry_points(torch, api):
    """sparc_gpu_gram / sparc_gpu_rotate_rows on a row block with an odd row count and padded leading dimensions."""
    wl = wlmod.make_workload(0)
    g = api.SparcGpu(wl)
    rng = np.random.default_rng(11)
    nr, m, n = 1237, 9, 5
    A, B = rng.standard_normal((nr, m)), rng.standard_normal((nr, n))
    Ad, Bd = api.colmajor_from_numpy(A, ld=nr + 3), api.colmajor_from_numpy(B, ld=nr + 1)
    G = api.colmajor_to_numpy(g.gram(Ad, Bd, nr))
    assert fro(G, orc.gram(A, B)) <= 1e-13
    S = api.colmajor_to_numpy(g.gram(Ad, Ad, nr, symmetric=True))
    assert fro(S, orc.gram(A, A)) <= 1e-13 and np.array_equal(S, S.T)
    Q = rng.standard_normal((m, m))
    g.rotate_rows(Ad, nr, api.colmajor_from_numpy(Q), row_panel=500)
    assert fro(api.colmajor_to_numpy(Ad, nr), orc.rotate(A, Q)) <= 1e-13
    with pytest.raises(api.SparcGpuError):
        g.gram(Ad, Bd, nr, symmetric=True)           # symmetric needs m = n
    # a rank that owns no rows: empty blocks (NULL data pointers), no workspace -> C = 0, through the C ABI itself
    import ctypes as C
    Cz = torch.full((n, m), 3.0, dtype=torch.float64, device="cuda:0")
    null = C.c_void_p(0)
    rc = g.lib.sparc_gpu_gram(g._ctx, null, 0, null, 0, 0, m, n, C.c_void_p(Cz.data_ptr()), 0, null,
                              C.c_void_p(torch.cuda.current_stream().cuda_stream))
    torch.cuda.synchronize()
    assert rc == 0 and float(Cz.abs().max()) == 0.0
    E = torch.empty((m, 0), dtype=torch.float64, device="cuda:0")
    assert float(g.gram(E, E, 0, symmetric=True).abs().max()) == 0.0
    g.close()
