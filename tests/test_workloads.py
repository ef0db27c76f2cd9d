"""The seeded input generator (paper_2302_09708_b200/workloads.py): determinism, structure, sizes."""
import numpy as np
import pytest

from paper_2302_09708_b200 import workloads as wlmod


def test_counter_uniform_is_stateless_and_in_range():
    u = wlmod.counter_uniform(3, 1, np.arange(1000))
    v = wlmod.counter_uniform(3, 1, np.arange(500, 1000))
    assert np.array_equal(u[500:], v)
    assert u.min() >= 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 0.05
    assert not np.array_equal(u, wlmod.counter_uniform(3, 2, np.arange(1000)))
    assert not np.array_equal(u, wlmod.counter_uniform(4, 1, np.arange(1000)))
    # scalar python restatement of the same mix (guards the uint64 wrap-around arithmetic)
    key = wlmod.stream_key(3, 1)
    z = wlmod._mix64_int(key + wlmod._GOLDEN * 777)
    assert u[777] == (z >> 11) / 2.0 ** 53


@pytest.mark.parametrize("cfg,cov", [(0, 0.27), (1, 0.52)])
def test_named_workloads_shapes(cfg, cov):
    wl = wlmod.make_workload(cfg)
    c = wlmod.CONFIG_TABLE[cfg]
    assert wl.nd == c["n"][0] * c["n"][1] * c["n"][2]
    assert wl.n_atoms == c["atoms"] and int(wl.n_proj[0]) == c["P"]
    assert abs(wl.coverage - cov) < 0.06                       # SURVEY.md section 8 size table
    assert wl.a0 < wl.a < wl.b
    assert wl.veff.shape == (wl.nd,)
    for J in range(wl.n_atoms):
        idx = wl.supp_idx[wl.supp_ptr[J]:wl.supp_ptr[J + 1]]
        assert np.all(np.diff(idx) > 0) and idx.min() >= 0 and idx.max() < wl.nd
        assert wl.chi_ptr[J + 1] - wl.chi_ptr[J] == idx.size * wl.n_proj[J]
    # same seed -> same data
    wl2 = wlmod.make_workload(cfg)
    assert np.array_equal(wl.chi, wl2.chi) and np.array_equal(wl.veff, wl2.veff)
    p = wl.psi_columns([0, 3])
    assert p.shape == (wl.nd, 2) and np.abs(p).max() <= 1.0
    assert np.array_equal(p[:, 1], wl.psi_columns([3])[:, 0])


def test_q_is_orthogonal():
    wl = wlmod.make_workload(0)
    Q = wl.q_matrix()
    assert Q.shape == (32, 32)
    assert np.max(np.abs(Q.T @ Q - np.eye(32))) < 1e-13
    assert np.max(np.abs(Q - Q.T)) > 1e-2


def test_slab_support_respects_dirichlet_faces():
    # an atom near a Dirichlet face loses the part of its support outside the grid; near a periodic
    # face the support wraps
    n, h = (16, 16, 16), (0.5, 0.5, 0.5)
    pos = np.array([[0.1, 4.0, 0.2]])
    wl = wlmod.make_custom("s", n, h, (0, 0, 1), 1, 1, pos, [4], 2.0)
    idx = wl.supp_idx.astype(np.int64)
    x, z = idx % 16, idx // 256
    assert x.max() == 15 and x.min() == 0          # wrapped in x
    assert z.max() <= 4                            # cut in z, not wrapped
    full = wlmod.make_custom("s", n, h, (0, 0, 0), 1, 1, pos, [4], 2.0)
    assert full.supp_idx.size > wl.supp_idx.size
