"""Bounds and race checks of our own (compute-sanitizer is closed on this GPU pool): every operator of
the hot path runs with sentinel-filled guard bands in front of and behind Psi, the outputs and the workspace, and in the
padding rows [N_d, ld) of every column; afterwards every guard byte must be intact (a stray store of a tile tail, a halo
plane, a slab of the bulk reduce-add or a split-K partial would land there).  The race-prone kernels are then repeated from
the same input: the paths with a fixed summation order (stencil, project + pull nonlocal mode, GEMMs, in-place rotation by row
panels) must give identical bits every time, the brick kernel (order of its reduce-adds is free) the same numbers to
rounding.  Parity with the CPU oracle is what the other GPU tests check; here only what the oracle cannot see."""
import numpy as np
import pytest

from paper_2302_09708_b200 import workloads as wlmod

pytestmark = pytest.mark.gpu

SENTINEL = -0x0123456789ABCDF       # an int64 pattern no kernel produces (as a double: a large negative normal number)
GUARD = 1 << 16                     # int64 words per guard band (512 KiB)


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


@pytest.fixture(scope="module")
def api():
    from paper_2302_09708_b200 import api as a
    return a


class Guarded:
    """A float64 (ncols, ld) matrix, or a byte workspace, cut out of a sentinel-filled buffer with a guard band on each side."""

    def __init__(self, torch, ncols, ld, nd):
        self.torch, self.ncols, self.ld, self.nd = torch, ncols, ld, nd
        self.raw = torch.full((2 * GUARD + ncols * ld,), SENTINEL, dtype=torch.int64, device="cuda:0")
        self.mat = self.raw[GUARD:GUARD + ncols * ld].view(torch.float64).view(ncols, ld)

    def bytes(self):
        return self.raw[GUARD:GUARD + self.ncols * self.ld].view(self.torch.uint8)

    def intact(self):
        r = self.raw
        ok = bool((r[:GUARD] == SENTINEL).all()) and bool((r[GUARD + self.ncols * self.ld:] == SENTINEL).all())
        if self.ld > self.nd:       # padding rows of every column
            pad = r[GUARD:GUARD + self.ncols * self.ld].view(self.ncols, self.ld)[:, self.nd:]
            ok = ok and bool((pad == SENTINEL).all())
        return ok


def _ragged():
    pos = np.array([[1.0, 2.0, 3.0], [5.5, 5.0, 0.4], [3.0, 0.2, 6.0]])
    return wlmod.make_custom("guard_ragged", (24, 18, 17), (0.4, 0.45, 0.5), (0, 1, 0), 37, 5, pos, [9, 4, 1], 2.6, seed=23)


@pytest.mark.parametrize("case", ["cfg0", "cfg1", "ragged"])
@pytest.mark.parametrize("nl_mode", [0, 1])
def test_no_store_outside_the_buffers_and_repeatable_bits(torch, api, case, nl_mode):
    wl = wlmod.make_workload(0) if case == "cfg0" else wlmod.make_workload(1) if case == "cfg1" else _ragged()
    ns, nd = wl.ns, wl.nd
    ld = nd + 16
    g = api.SparcGpu(wl)
    g.set_option("nonlocal_mode", nl_mode)
    col_block = 0 if case != "ragged" else 16
    row_panel = 0 if case != "ragged" else 1000
    need = max(g.workspace_bytes(op, ns, blk) for op, blk in ((api.OP_HAMILTONIAN_APPLY, 0), (api.OP_CHEBYSHEV_FILTER, col_block),
                                                              (api.OP_PROJECT, col_block), (api.OP_ROTATE, row_panel)))
    words = (need + 7) // 8
    ws = Guarded(torch, 1, words, words)
    g._ws = ws.bytes()                                   # the binding uses (and declares) this buffer as ws_dev
    assert g.lib.sparc_gpu_set_workspace_size(g._ctx, g._ws.numel()) == 0 and g._ws.data_ptr() % 256 == 0

    psi0 = torch.empty((ns, nd), dtype=torch.float64, device="cuda:0")
    api.fill_uniform(psi0, wl.seed, wlmod.STREAM_PSI, 0, -1.0, 1.0)
    Q = api.colmajor_from_numpy(np.linalg.qr(np.random.default_rng(3).standard_normal((ns, ns)))[0])
    X, Y = Guarded(torch, ns, ld, nd), Guarded(torch, ns, ld, nd)
    Hs, Ms = Guarded(torch, ns, ns, ns), Guarded(torch, ns, ns, ns)

    def one_pass():
        X.mat[:, :nd] = psi0
        g.hamiltonian_apply(X.mat, Y.mat)
        y = Y.mat[:, :nd].clone()
        g.chebyshev_filter(X.mat, wl.degree, wl.a, wl.b, wl.a0, col_block=col_block)
        f = X.mat[:, :nd].clone()
        g.project(X.mat, col_block=col_block, Hs=Hs.mat, Ms=Ms.mat)
        h, m = Hs.mat.clone(), Ms.mat.clone()
        g.rotate(X.mat, Q, row_panel=row_panel)
        r = X.mat[:, :nd].clone()
        torch.cuda.synchronize()
        return y, f, h, m, r

    runs = [one_pass() for _ in range(3)]
    for name, buf in (("Psi", X), ("Y", Y), ("Hs", Hs), ("Ms", Ms), ("workspace", ws)):
        assert buf.intact(), f"{case}, nonlocal_mode {nl_mode}: a kernel wrote outside {name} (guard band or padding rows)"
    brick = nl_mode == 0 and g.get_info("nl_brick") == 1
    names = ("H*Psi", "filter", "Hs", "Ms", "Psi*Q")
    for k in (1, 2):
        for name, a, b in zip(names, runs[0], runs[k]):
            assert bool(torch.isfinite(b).all())
            if brick:       # reduce-adds in free order: equal to rounding
                err = float((a - b).norm() / a.norm())
                assert err <= 1e-13, f"{case}: {name} differs between identical runs by {err:.2e}"
            else:
                assert torch.equal(a, b), f"{case}, nonlocal_mode {nl_mode}: {name} is not bitwise repeatable"
    # rotation and projection alone are fixed-order whatever the nonlocal path: same input, same bits
    X.mat[:, :nd] = runs[0][1]
    g.project(X.mat, col_block=col_block, Hs=Hs.mat, Ms=Ms.mat)
    m1 = Ms.mat.clone()
    g.rotate(X.mat, Q, row_panel=row_panel)
    r1 = X.mat[:, :nd].clone()
    X.mat[:, :nd] = runs[0][1]
    g.project(X.mat, col_block=col_block, Hs=Hs.mat, Ms=Ms.mat)
    g.rotate(X.mat, Q, row_panel=row_panel)
    torch.cuda.synchronize()
    assert torch.equal(m1, Ms.mat) and torch.equal(r1, X.mat[:, :nd])
    print(f"[guard] {case}, nonlocal_mode {nl_mode}: guards intact (workspace {need >> 20} MiB), stencil path "
          f"{g.get_info('stencil_path_last')}, brick {int(brick)}, 3 identical runs")
    g._ws = None
    g.close()
