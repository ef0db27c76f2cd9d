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
