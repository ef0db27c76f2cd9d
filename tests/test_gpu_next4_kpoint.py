"""GPU parity: the complex (k-point) operators -- H(k) X with Bloch phases on the periodic
wraps and on the projector images, the Chebyshev filter, the Hermitian products Hs = Psi^H H Psi, Ms = Psi^H Psi and the
complex rotation -- CUDA path through the C ABI against oracle/chefsi_next_oracle.c
(K1-K4), element by element, same gates as the real path (1e-10 per column, 1e-11 Frobenius; tight 1e-13)."""
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


def fro_err(G, O):
    return float(np.linalg.norm(G - O) / np.linalg.norm(O))


def to_dev(torch, X, ld=None):
    """(rows x cols) complex numpy -> (cols, ld) complex128 CUDA tensor holding it column-major."""
    rows, cols = X.shape
    ld = rows if ld is None else ld
    t = torch.zeros((cols, ld), dtype=torch.complex128, device="cuda")
    t[:, :rows] = torch.from_numpy(np.ascontiguousarray(X.T)).cuda()
    return t


def to_host(t, rows=None):
    rows = t.shape[1] if rows is None else rows
    return np.asfortranarray(t[:, :rows].cpu().numpy().T)


def cases():
    out = []
    pos = np.array([[0.2, 3.1, 3.0], [3.6, 0.3, 0.4]])       # supports cross periodic faces: image shifts +-1 present
    for bc in [(0, 0, 0), (0, 0, 1), (1, 0, 0), (1, 1, 1)]:
        out.append((wlmod.make_custom(f"k_{bc}", (13, 14, 15), (0.5, 0.45, 0.4), bc, 5, 6, pos, [4, 9], 2.3, seed=41),
                    np.array([0.7, -1.9, 0.4])))
    pos2 = np.array([[1.0, 2.0, 3.0], [5.5, 5.0, 0.4], [3.0, 0.2, 6.0]])
    out.append((wlmod.make_custom("k_even", (24, 18, 17), (0.4, 0.45, 0.5), (0, 0, 0), 7, 5, pos2, [9, 4, 1], 2.6, seed=42),
                np.array([np.pi, 0.0, -2.5])))
    return out


@pytest.mark.parametrize("wl,theta", cases(), ids=lambda v: getattr(v, "name", None))
def test_hk_apply_filter_project_rotate(torch, api, wl, theta):
    g = api.SparcGpu(wl)
    g.set_kpoint(theta, wl.supp_shift)
    Hk = orc.HamiltonianK(wl, theta)
    X = wl.psi_columns_complex(range(wl.ns))
    ld = wl.nd + 3
    Xg = to_dev(torch, X, ld)
    Y = to_host(g.hamiltonian_apply_k(Xg), wl.nd)
    e = col_err(Y, Hk.apply(X))
    print(f"[parity] {wl.name} H(k) X: {e:.2e}")
    assert e <= 1e-10 and e <= 1e-13
    assert np.array_equal(to_host(Xg, wl.nd), X)
    for m in (1, 2, wl.degree):
        Pg = to_dev(torch, X, ld)
        g.chebyshev_filter_k(Pg, m, wl.a, wl.b, wl.a0, col_block=3)
        e = col_err(to_host(Pg, wl.nd), Hk.chebyshev_filter(X, m, wl.a, wl.b, wl.a0))
        print(f"[parity] {wl.name} filter_k m={m}: {e:.2e}")
        assert e <= 1e-10 and e <= 1e-13
    # subspace products and rotation on the filtered block of the oracle
    F = Hk.chebyshev_filter(X, wl.degree, wl.a, wl.b, wl.a0)
    Fg = to_dev(torch, F, ld)
    for cb in (0, 2):
        Hs, Ms = g.project_k(Fg, col_block=cb)
        Hs_o, Ms_o = orc.gram_k(F, Hk.apply(F)), orc.gram_k(F, F)
        e_h, e_m = fro_err(to_host(Hs), Hs_o), fro_err(to_host(Ms), Ms_o)
        print(f"[parity] {wl.name} project_k (col_block {cb}): Hs {e_h:.2e}, Ms {e_m:.2e}")
        assert max(e_h, e_m) <= 1e-11 and max(e_h, e_m) <= 1e-13
    Hh = to_host(Hs)
    assert np.max(np.abs(Hh - Hh.conj().T)) <= 1e-12 * np.max(np.abs(Hh))       # Hermitian up to rounding
    rng = np.random.default_rng(9)
    Q = rng.normal(size=(wl.ns, wl.ns)) + 1j * rng.normal(size=(wl.ns, wl.ns))    # not Hermitian: Q, Q^T, Q^H, conj(Q) differ
    for rp in (0, 1000):
        Rg = to_dev(torch, F, ld)
        g.rotate_k(Rg, to_dev(torch, Q), row_panel=rp)
        e = fro_err(to_host(Rg, wl.nd), orc.rotate_k(F, Q))
        print(f"[parity] {wl.name} rotate_k (row_panel {rp}): {e:.2e}")
        assert e <= 1e-11 and e <= 1e-13
    g.close()


def test_gamma_point_limit_and_kpoint_switch(torch, api):
    """theta = 0 with real input reproduces the real operator bit for bit in the imaginary part (zero); a second
    set_kpoint on the same context replaces the first."""
    pos = np.array([[1.0, 2.0, 3.0]])
    wl = wlmod.make_custom("k_gamma", (14, 13, 15), (0.5, 0.45, 0.4), (0, 1, 0), 3, 5, pos, [4], 2.0, seed=43)
    g = api.SparcGpu(wl)
    X = wl.psi_columns(range(3))
    g.set_kpoint((0.0, 0.0, 0.0), wl.supp_shift)
    Y0 = to_host(g.hamiltonian_apply_k(to_dev(torch, X.astype(complex))))
    Yr = orc.Hamiltonian(wl).apply(X)
    assert np.max(np.abs(Y0.imag)) == 0.0 and col_err(Y0.real, Yr) <= 1e-13
    theta = (1.1, 0.3, -0.6)
    g.set_kpoint(theta, wl.supp_shift)
    Xc = wl.psi_columns_complex(range(3))
    Y1 = to_host(g.hamiltonian_apply_k(to_dev(torch, Xc)))
    assert col_err(Y1, orc.HamiltonianK(wl, theta).apply(Xc)) <= 1e-13
    # a set_kpoint that fails validation (image shift outside -1..1) leaves the previous k-point fully in place
    bad = np.array(wl.supp_shift, dtype=np.int8).copy()
    bad[-1, 2] = 2
    with pytest.raises(api.SparcGpuError) as ei:
        g.set_kpoint((0.2, 0.2, 0.2), bad)
    assert ei.value.code == -4
    Y2 = to_host(g.hamiltonian_apply_k(to_dev(torch, Xc)))
    assert np.array_equal(Y1, Y2)
    # calls before any set_kpoint are refused
    g2 = api.SparcGpu(wl)
    with pytest.raises(api.SparcGpuError) as ei:
        g2.hamiltonian_apply_k(to_dev(torch, Xc))
    assert ei.value.code == -1
    g.close()
    g2.close()


def test_kpoint_config1_sampled(torch, api):
    """configs[1]'s grid and atoms (48^3, 32 atoms) with a complex block of 64 orbitals at k = (1/4, 1/4, 1/4) of the
    Brillouin zone: filter (degree 20) on the device, sampled columns against the oracle; Hermitian products on sampled
    entries; rotation on sampled rows."""
    wl = wlmod.make_workload(1)
    ns = 64
    theta = np.array([0.5 * np.pi] * 3)
    g = api.SparcGpu(wl)
    g.set_kpoint(theta, wl.supp_shift)
    X = wl.psi_columns_complex(range(ns))
    Pg = to_dev(torch, X)
    g.chebyshev_filter_k(Pg, wl.degree, wl.a, wl.b, wl.a0)
    Hk = orc.HamiltonianK(wl, theta)
    cols = [0, 31, 63]
    Fo = Hk.chebyshev_filter(X[:, cols], wl.degree, wl.a, wl.b, wl.a0)
    Fg = to_host(Pg)
    e = col_err(Fg[:, cols], Fo)
    print(f"[parity] cfg1 k-point filter, sampled columns: {e:.2e}")
    assert e <= 1e-10 and e <= 1e-13
    Hs, Ms = g.project_k(Pg)
    Hs_o = orc.gram_k(Fg[:, cols], Hk.apply(Fg[:, cols]))
    Ms_o = orc.gram_k(Fg[:, cols], Fg[:, cols])
    assert fro_err(to_host(Hs)[np.ix_(cols, cols)], Hs_o) <= 1e-11
    assert fro_err(to_host(Ms)[np.ix_(cols, cols)], Ms_o) <= 1e-11
    rng = np.random.default_rng(3)
    Q = np.linalg.qr(rng.normal(size=(ns, ns)) + 1j * rng.normal(size=(ns, ns)))[0]
    g.rotate_k(Pg, to_dev(torch, Q))
    rows = np.array([0, 1, 5000, 48 ** 3 - 1])
    Ro = orc.rotate_k(Fg[rows, :], Q)
    assert fro_err(to_host(Pg)[rows, :], Ro) <= 1e-11
    g.close()


def test_kpoint_config2_grid_256_orbitals_sampled(torch, api):
    """configs[2]'s grid and atoms (60 x 60 x 180 slab, Dirichlet z) with 256 complex orbitals, the block generated on the
    device (same counter-based generator as the host's): filter on sampled columns, Hermitian products on sampled entries and
    the rotation on sampled rows against the oracle -- the k-point path at a size where the column blocking, the real-view
    GEMMs and the row panels all take several tiles."""
    wl = wlmod.make_workload(2)
    ns, nd = 256, wl.nd
    theta = np.array([0.5 * np.pi, 0.25 * np.pi, 0.0])
    g = api.SparcGpu(wl)
    g.set_kpoint(theta, wl.supp_shift)
    re = torch.empty((ns, nd), dtype=torch.float64, device="cuda")
    im = torch.empty_like(re)
    api.fill_uniform(re, wl.seed, wlmod.STREAM_PSI, 0, -1.0, 1.0)
    api.fill_uniform(im, wl.seed, wlmod.STREAM_PSI_IMAG, 0, -1.0, 1.0)
    Pg = torch.complex(re, im)
    del re, im
    cols = [0, 100, 255]
    X = wl.psi_columns_complex(cols)
    assert np.array_equal(to_host(Pg[cols]), X)               # the two generators agree bit for bit
    g.chebyshev_filter_k(Pg, wl.degree, wl.a, wl.b, wl.a0)
    Hk = orc.HamiltonianK(wl, theta)
    Fo = Hk.chebyshev_filter(X, wl.degree, wl.a, wl.b, wl.a0)
    Fg = to_host(Pg[cols])
    e = col_err(Fg, Fo)
    print(f"[parity] cfg2-grid k-point filter, 256 orbitals, sampled columns: {e:.2e}")
    assert e <= 1e-10 and e <= 1e-13
    Hs, Ms = g.project_k(Pg)
    Hs_o = orc.gram_k(Fg, Hk.apply(Fg))
    Ms_o = orc.gram_k(Fg, Fg)
    assert fro_err(to_host(Hs)[np.ix_(cols, cols)], Hs_o) <= 1e-11
    assert fro_err(to_host(Ms)[np.ix_(cols, cols)], Ms_o) <= 1e-11
    rows = np.array([0, 59, 3600, 300000, nd - 1])
    before = np.ascontiguousarray(Pg[:, torch.from_numpy(rows).cuda()].cpu().numpy().T)      # (rows, ns)
    rng = np.random.default_rng(4)
    Q = np.linalg.qr(rng.normal(size=(ns, ns)) + 1j * rng.normal(size=(ns, ns)))[0]
    g.rotate_k(Pg, to_dev(torch, Q))
    after = np.ascontiguousarray(Pg[:, torch.from_numpy(rows).cuda()].cpu().numpy().T)
    assert fro_err(after, orc.rotate_k(before, Q)) <= 1e-11
    g.close()


def test_kpoint_lower_fd_order(torch, api):
    """FD order 4 (radius 2) on a short periodic grid: wrapped taps with their phases for a stencil narrower than the maximum."""
    pos = np.array([[1.0, 2.0, 1.5]])
    wl = wlmod.make_custom("k_fd4", (7, 9, 8), (0.5, 0.45, 0.4), (0, 0, 1), 3, 4, pos, [4], 1.2, seed=45, fd_order=4)
    theta = np.array([2.1, -0.8, 0.3])
    g = api.SparcGpu(wl)
    g.set_kpoint(theta, wl.supp_shift)
    X = wl.psi_columns_complex(range(wl.ns))
    Hk = orc.HamiltonianK(wl, theta)
    assert col_err(to_host(g.hamiltonian_apply_k(to_dev(torch, X))), Hk.apply(X)) <= 1e-13
    Pg = to_dev(torch, X)
    g.chebyshev_filter_k(Pg, 3, wl.a, wl.b, wl.a0)
    assert col_err(to_host(Pg), Hk.chebyshev_filter(X, 3, wl.a, wl.b, wl.a0)) <= 1e-13
    g.close()
