"""GPU parity of the host-buffer entry point sparc_gpu_chefsi_step_host (whole step: filter -> project -> rotate with the
PCIe copies overlapped) against the CPU oracle, same gates as tests/test_gpu_parity.py."""
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


def fro_err(G, O):
    return float(np.linalg.norm(G - O) / np.linalg.norm(O))


@pytest.mark.parametrize("case", ["cfg0", "ragged"])
def test_step_host_matches_oracle(torch, api, case):
    if case == "cfg0":
        wl = wlmod.make_workload(0)
        col_block, row_panel, pad = 0, 0, 0
    else:       # odd column count, chunks with a ragged tail, padded host leading dimension, several row panels
        pos = np.array([[1.0, 2.0, 3.0], [5.5, 5.0, 0.4], [3.0, 0.2, 6.0]])
        wl = wlmod.make_custom("step_host_ragged", (24, 18, 17), (0.4, 0.45, 0.5), (0, 1, 0), 71, 5, pos, [9, 4, 1], 2.6, seed=21)
        col_block, row_panel, pad = 16, 1000, 10
    ns, nd = wl.ns, wl.nd
    X = wl.psi_columns(range(ns))
    rng = np.random.default_rng(5)
    Q = np.linalg.qr(rng.standard_normal((ns, ns)))[0]
    H = orc.Hamiltonian(wl)
    F = H.chebyshev_filter(X, wl.degree, wl.a, wl.b, wl.a0)
    Hs_o, Ms_o = H.project(F)
    R_o = orc.rotate(F, Q)

    g = api.SparcGpu(wl)
    ld = nd + pad
    host = torch.zeros((ns, ld), dtype=torch.float64).pin_memory()
    host[:, :nd] = torch.from_numpy(np.ascontiguousarray(X.T))
    Qh = torch.from_numpy(np.ascontiguousarray(Q.T)).pin_memory()
    Hs = torch.empty((ns, ns), dtype=torch.float64).pin_memory()
    Ms = torch.empty((ns, ns), dtype=torch.float64).pin_memory()
    launches0 = g.get_info("kernel_launches")
    g.chefsi_step_host(host, Qh, Hs, Ms, wl.degree, wl.a, wl.b, wl.a0, col_block=col_block, row_panel=row_panel)
    assert g.get_info("kernel_launches") > launches0
    G = host[:, :nd].numpy().T
    e_r, e_h, e_m = fro_err(G, R_o), fro_err(Hs.numpy().T, Hs_o), fro_err(Ms.numpy().T, Ms_o)
    print(f"[parity] step_host {case}: Psi Q {e_r:.2e}, Hs {e_h:.2e}, Ms {e_m:.2e}")
    assert max(e_r, e_h, e_m) <= 1e-11
    assert max(e_r, e_h, e_m) <= 1e-13
    if pad:
        assert float(host[:, nd:].abs().max()) == 0.0          # the padding rows of the host block are not written

    # separate output buffer; bad bounds and a short workspace are error codes
    host2 = torch.zeros((ns, ld), dtype=torch.float64).pin_memory()
    host2[:, :nd] = torch.from_numpy(np.ascontiguousarray(X.T))
    out = torch.zeros_like(host2).pin_memory()
    g.chefsi_step_host(host2, Qh, Hs, Ms, wl.degree, wl.a, wl.b, wl.a0, col_block=col_block, row_panel=row_panel, host_out=out)
    assert fro_err(out[:, :nd].numpy().T, R_o) <= 1e-13
    assert np.array_equal(host2[:, :nd].numpy().T, X)
    with pytest.raises(api.SparcGpuError) as ei:
        g.chefsi_step_host(host2, Qh, Hs, Ms, wl.degree, wl.b, wl.a, wl.a0)
    assert ei.value.code == -3
    g.close()


@pytest.mark.parametrize("case", ["cfg0", "ragged"])
def test_step_host_solve_is_algorithm_1(torch, api, case):
    """sparc_gpu_chefsi_step_host_solve: filter -> project -> device eigensolve -> rotate with no Q from the caller
    (PAPER.md:41-45, 79-84).  Hs, Ms against the oracle; D against the oracle's generalized eigenvalues; the returned block
    spans the filtered block, is M-orthonormal and makes Hs diagonal with D on the diagonal (Z itself is unique only up to
    signs and rotations inside degenerate eigenspaces, reading R23, so it is not compared entry-wise)."""
    if case == "cfg0":
        wl = wlmod.make_workload(0)
        col_block, row_panel, pad = 0, 0, 0
    else:
        pos = np.array([[1.0, 2.0, 3.0], [5.5, 5.0, 0.4], [3.0, 0.2, 6.0]])
        wl = wlmod.make_custom("step_host_ragged", (24, 18, 17), (0.4, 0.45, 0.5), (0, 1, 0), 71, 5, pos, [9, 4, 1], 2.6, seed=21)
        col_block, row_panel, pad = 16, 1000, 10
    ns, nd = wl.ns, wl.nd
    X = wl.psi_columns(range(ns))
    H = orc.Hamiltonian(wl)
    F = H.chebyshev_filter(X, wl.degree, wl.a, wl.b, wl.a0)
    Hs_o, Ms_o = H.project(F)
    D_o, _ = orc.sygv(0.5 * (Hs_o + Hs_o.T), Ms_o)

    g = api.SparcGpu(wl)
    ld = nd + pad
    host = torch.zeros((ns, ld), dtype=torch.float64).pin_memory()
    host[:, :nd] = torch.from_numpy(np.ascontiguousarray(X.T))
    Hs = torch.empty((ns, ns), dtype=torch.float64).pin_memory()
    Ms = torch.empty((ns, ns), dtype=torch.float64).pin_memory()
    launches0 = g.get_info("kernel_launches")
    out, D, info = g.chefsi_step_host_solve(host, Hs, Ms, wl.degree, wl.a, wl.b, wl.a0, col_block=col_block, row_panel=row_panel)
    assert g.get_info("kernel_launches") > launches0
    assert int(info[0]) == 0 and int(info[1]) >= 1
    e_h, e_m = fro_err(Hs.numpy().T, Hs_o), fro_err(Ms.numpy().T, Ms_o)
    Dn = D.numpy()
    scale = max(1.0, float(np.abs(D_o).max()))
    e_d = float(np.max(np.abs(Dn - D_o))) / scale
    G = np.ascontiguousarray(out[:, :nd].numpy().T)
    Hs2, Ms2 = H.project(G)
    # conditioning: a filtered random block is far from orthonormal, so the gates of the rotated block scale with cond(Ms)
    cond = float(np.linalg.cond(Ms_o))
    e_i = float(np.max(np.abs(Ms2 - np.eye(ns))))
    e_g = float(np.max(np.abs(Hs2 - np.diag(Dn)))) / scale
    coef = np.linalg.lstsq(F, G, rcond=None)[0]
    e_s = fro_err(F @ coef, G)
    print(f"[parity] step_host_solve {case}: Hs {e_h:.2e}, Ms {e_m:.2e}, D {e_d:.2e}, Z^T Ms Z - I {e_i:.2e}, "
          f"Z^T Hs Z - D {e_g:.2e}, span {e_s:.2e}, cond(Ms) {cond:.1e}, sweeps {int(info[1])}")
    assert max(e_h, e_m) <= 1e-13
    assert e_d <= 1e-11 * max(1.0, cond * 1e-4)
    assert e_i <= 1e-14 * max(1e3, cond) and e_g <= 1e-14 * max(1e3, cond)
    assert e_s <= 1e-10
    if pad:
        assert float(out[:, nd:].abs().max()) == 0.0
    # the solving variant needs its two extra outputs; the plain entry point still refuses a missing Q
    import ctypes as C
    lib = api.load_library()
    null = C.c_void_p(0)
    p = C.c_void_p(host.data_ptr())
    assert lib.sparc_gpu_chefsi_step_host_solve(g._ctx, p, p, ld, ns, wl.degree, wl.a, wl.b, wl.a0, null, null, p, p, p, ld, p,
                                                0, 0, p, null) == -1
    assert lib.sparc_gpu_chefsi_step_host(g._ctx, p, p, ld, ns, wl.degree, wl.a, wl.b, wl.a0, null, p, p, p, ld, p,
                                          0, 0, p, null) == -1
    g.close()
