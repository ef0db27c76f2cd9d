"""GPU parity: gradient stencil, projector contraction chi^T X and the nonlocal force
(PAPER.md:110, 188), CUDA path through the C ABI against oracle/chefsi_next_oracle.c (G2-G4), element by element.
Gates: gradient like H*Psi (max |d| / ||column||_2 <= 1e-10, tight 1e-13); W and F relative (Frobenius / max) <= 1e-11."""
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


def col_err(G, O):
    return float((np.max(np.abs(G - O), axis=0) / np.linalg.norm(O, axis=0)).max())


def cases():
    pos = np.array([[0.2, 3.1, 3.3], [4.1, 6.2, 0.7]])
    out = []
    for bc in [(0, 0, 0), (1, 1, 1), (0, 1, 0), (1, 0, 1)]:
        out.append(wlmod.make_custom(f"g_odd_{bc}", (13, 14, 19), (0.5, 0.45, 0.4), bc, 5, 4, pos, [4, 9], 2.5, seed=31))
    pos2 = np.array([[1.0, 2.0, 3.0], [5.5, 5.0, 0.4], [3.0, 0.2, 6.0]])
    for bc in [(0, 0, 0), (0, 0, 1)]:      # several chunks per axis with ragged tails (x: 4, y / z: 16 outputs per thread)
        out.append(wlmod.make_custom(f"g_even_{bc}", (26, 35, 41), (0.4, 0.45, 0.5), bc, 7, 4, pos2, [9, 4, 1], 2.6, seed=32))
    return out


@pytest.mark.parametrize("wl", cases(), ids=lambda w: w.name)
def test_gradient_project_force_small(torch, api, wl):
    g = api.SparcGpu(wl)
    F = orc.Forces(wl)
    X = wl.psi_columns(range(wl.ns))
    ld = wl.nd + 5
    Xg = api.colmajor_from_numpy(X, ld=ld)
    for axis in range(3):
        Yg = g.gradient(Xg, axis)
        e = col_err(api.colmajor_to_numpy(Yg, wl.nd), F.gradient(X, axis))
        print(f"[parity] {wl.name} gradient axis {axis}: {e:.2e}")
        assert e <= 1e-10 and e <= 1e-13
        Wo = F.nl_project(F.gradient(X, axis))
        Wg = g.gradient_project(Xg, axis, col_block=3).cpu().numpy().T
        assert np.linalg.norm(Wg - Wo) <= 1e-13 * np.linalg.norm(Wo)
    assert np.array_equal(api.colmajor_to_numpy(Xg, wl.nd), X)
    Wo = F.nl_project(X)
    Wg = g.nl_project(Xg).cpu().numpy().T
    assert np.linalg.norm(Wg - Wo) <= 1e-13 * np.linalg.norm(Wo)
    occ = wl.occupations()
    Fo = F.nonlocal_force(X, occ)
    occ_g = torch.from_numpy(occ).cuda()
    for cb in (0, 2):                                      # column blocking must not matter (R19)
        Fg = g.nonlocal_force(Xg, occ_g, col_block=cb).cpu().numpy()
        e = float(np.max(np.abs(Fg - Fo)) / np.max(np.abs(Fo)))
        print(f"[parity] {wl.name} force (col_block {cb}): {e:.2e}")
        assert e <= 1e-11
    # bitwise reproducible
    assert np.array_equal(g.nonlocal_force(Xg, occ_g, col_block=2).cpu().numpy(), Fg)
    g.close()


def test_lower_orders_and_degenerate(torch, api):
    pos = np.array([[1.0, 2.0, 3.0]])
    for fd_order in (2, 6):
        wl = wlmod.make_custom(f"g_fd{fd_order}", (9, 8, 7), (0.5, 0.5, 0.5), (0, 1, 0), 3, 2, pos, [4], 1.5, seed=33,
                               fd_order=fd_order)
        g = api.SparcGpu(wl)
        F = orc.Forces(wl)
        X = wl.psi_columns(range(wl.ns))
        Xg = api.colmajor_from_numpy(X)
        for axis in range(3):
            assert col_err(api.colmajor_to_numpy(g.gradient(Xg, axis), wl.nd), F.gradient(X, axis)) <= 1e-13
        g.close()
    wl = wlmod.make_custom("g_noatoms", (14, 14, 14), (0.5,) * 3, (0, 0, 0), 2, 2, np.zeros((0, 3)), [], 2.0, seed=34)
    g = api.SparcGpu(wl)
    Xg = api.colmajor_from_numpy(wl.psi_columns(range(2)))
    assert g.nonlocal_force(Xg, torch.ones(2, dtype=torch.float64, device="cuda")).shape[0] == 0
    with pytest.raises(api.SparcGpuError) as ei:
        g.lib.sparc_gpu_gradient.restype = int
        api._check(g.lib.sparc_gpu_gradient(g._ctx, 3, None, 0, None, 0, 1, None), "gradient")
    assert ei.value.code == -1
    g.close()


def test_force_config1_full(torch, api):
    """Configs[1] at full size (48^3 x 256): the force on all 32 atoms, and chi^T D_a Psi on sampled columns."""
    wl = wlmod.make_workload(1)
    g = api.SparcGpu(wl)
    psi = torch.empty((wl.ns, wl.nd), dtype=torch.float64, device="cuda")
    api.fill_uniform(psi, wl.seed, wlmod.STREAM_PSI, 0, -1.0, 1.0)
    occ = wl.occupations()
    Fg = g.nonlocal_force(psi, torch.from_numpy(occ).cuda()).cpu().numpy()
    F = orc.Forces(wl)
    Fo = F.nonlocal_force(wl.psi(), occ)
    e = float(np.max(np.abs(Fg - Fo)) / np.max(np.abs(Fo)))
    print(f"[parity] cfg1 nonlocal force: {e:.2e}")
    assert e <= 1e-11
    cols = [0, 17, 255]
    Xc = wl.psi_columns(cols)
    for axis in range(3):
        Wg = g.gradient_project(psi, axis).cpu().numpy().T[:, cols]
        Wo = F.nl_project(F.gradient(Xc, axis))
        assert np.linalg.norm(Wg - Wo) <= 1e-12 * np.linalg.norm(Wo)
    g.close()
