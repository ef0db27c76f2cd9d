"""Pins of the CPU oracle (oracle/chefsi_oracle.c) against what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path.  Pin numbering follows DESIGN.md
section 4 (= SURVEY.md section 8(c)): P1 weights, P2 FD symbol on plane waves, P3 polynomial exactness,
P4 Dirichlet = restricted zero-padded periodic, P5 dense brute-force H + eigen-decomposition filter,
P6 symmetry, P7 T_m scaling / orthogonal-projector eigen relation, P8 small degrees, P9 column
independence, P10 Gram and rotation invariants.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2302_09708_b200 import workloads as wlmod


# ----------------------------------------------------------------------------- helpers
def golden_weights(golden_dir):
    w = {}
    with open(os.path.join(golden_dir, "fd_weights_r6.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            p, num, den = line.split()
            w[int(p)] = Fraction(int(num), int(den))
    return [w[p] for p in range(7)]


def cheb_T(m, t):
    """T_m(t) from its trigonometric / hyperbolic definition (independent of any recurrence)."""
    t = np.asarray(t, dtype=np.float64)
    out = np.empty_like(t)
    inside = np.abs(t) <= 1.0
    out[inside] = np.cos(m * np.arccos(t[inside]))
    tt = t[~inside]
    out[~inside] = np.sign(tt) ** m * np.cosh(m * np.arccosh(np.abs(tt)))
    return out


def empty_atoms_workload(n, h, bc, veff_kind="zero", ns=4, degree=6):
    return wlmod.make_custom("t", n, h, bc, ns, degree, np.zeros((0, 3)), np.zeros(0, np.int32), 3.0,
                             veff_kind=veff_kind)


def rand(shape, seed):
    return np.asfortranarray(np.random.default_rng(seed).uniform(-1, 1, size=shape))


# ----------------------------------------------------------------------------- P1
def test_P1_weights_match_rationals_and_moments(golden_dir):
    gw = golden_weights(golden_dir)
    w = orc.fd_weights(6)
    for p in range(7):
        assert abs(w[p] - float(gw[p])) <= 2e-16 * max(1.0, abs(float(gw[p])))
    # the rationals themselves: 12th-order accuracy conditions in exact arithmetic
    assert gw[0] + 2 * sum(gw[1:]) == 0
    assert 2 * sum(Fraction(p) ** 2 * gw[p] for p in range(1, 7)) == 2
    for j in range(2, 7):
        assert 2 * sum(Fraction(p) ** (2 * j) * gw[p] for p in range(1, 7)) == 0
    assert 2 * sum(Fraction(p) ** 14 * gw[p] for p in range(1, 7)) != 0
    # oracle doubles obey the same conditions to rounding
    assert abs(w[0] + 2 * w[1:].sum()) < 1e-14
    assert abs(2 * sum(p ** 2 * w[p] for p in range(1, 7)) - 2.0) < 1e-13


@pytest.mark.parametrize("radius,expect", [
    (1, [-2.0, 1.0]),
    (2, [-5.0 / 2, 4.0 / 3, -1.0 / 12]),
    (3, [-49.0 / 18, 3.0 / 2, -3.0 / 20, 1.0 / 90]),
])
def test_P1_low_order_textbook_weights(radius, expect):
    # textbook 2nd/4th/6th-order central second-derivative weights
    w = orc.fd_weights(radius)
    assert np.allclose(w, expect, rtol=0, atol=1e-15)


# ----------------------------------------------------------------------------- P2
def test_P2_symbol_spot_values(golden_dir):
    gw = [float(x) for x in golden_weights(golden_dir)]
    with open(os.path.join(golden_dir, "fd_symbol_spot.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            kh, val, tol = map(float, line.split())
            s = gw[0] + 2 * sum(gw[p] * math.cos(p * kh) for p in range(1, 7))
            assert abs(s - val) < tol


@pytest.mark.parametrize("n,h,modes", [
    ((16, 18, 20), (0.5, 0.45, 0.4), (1, 2, 3)),
    ((24, 24, 24), (0.5, 0.5, 0.5), (5, 0, 11)),
    ((13, 15, 14), (0.3, 0.7, 0.2), (6, 7, 1)),
])
def test_P2_plane_wave_symbol(golden_dir, n, h, modes):
    """L cos(k.r + phi) = [sum_axis (w0 + 2 sum_p w_p cos(p k h))/h^2] cos(k.r + phi) on a periodic grid."""
    gw = [float(x) for x in golden_weights(golden_dir)]
    wl = empty_atoms_workload(n, h, (0, 0, 0))
    H = orc.Hamiltonian(wl)
    k = [2 * math.pi * modes[a] / (n[a] * h[a]) for a in range(3)]
    x = np.arange(n[0]) * h[0]
    y = np.arange(n[1]) * h[1]
    z = np.arange(n[2]) * h[2]
    psi = np.cos(k[0] * x[None, None, :] + k[1] * y[None, :, None] + k[2] * z[:, None, None] + 0.3).ravel()
    sym = sum((gw[0] + 2 * sum(gw[p] * math.cos(p * k[a] * h[a]) for p in range(1, 7))) / h[a] ** 2
              for a in range(3))
    out = H.laplacian(psi)[:, 0]
    scale = abs(sym) * np.abs(psi).max() + 1.0
    assert np.max(np.abs(out - sym * psi)) / scale < 5e-13


# ----------------------------------------------------------------------------- P3
def test_P3_polynomial_exactness_interior():
    n, h = (16, 15, 14), (0.1, 0.12, 0.09)
    wl = empty_atoms_workload(n, h, (1, 1, 1))
    H = orc.Hamiltonian(wl)
    x = (np.arange(n[0]) * h[0])[None, None, :]
    y = (np.arange(n[1]) * h[1])[None, :, None]
    z = (np.arange(n[2]) * h[2])[:, None, None]
    f = x ** 12 + 2 * y ** 13 + z ** 11 * x + x ** 4 * y ** 4 * z ** 4 - 3 * x * y * z + 1.0
    lap = (132 * x ** 10 + 2 * 156 * y ** 11 + 110 * z ** 9 * x
           + 12 * x ** 2 * y ** 4 * z ** 4 + 12 * x ** 4 * y ** 2 * z ** 4 + 12 * x ** 4 * y ** 4 * z ** 2)
    f = np.broadcast_to(f, (n[2], n[1], n[0]))
    lap = np.broadcast_to(lap, (n[2], n[1], n[0]))
    out = H.laplacian(np.ascontiguousarray(f).ravel())[:, 0].reshape(n[2], n[1], n[0])
    inner = (slice(6, n[2] - 6), slice(6, n[1] - 6), slice(6, n[0] - 6))
    err = np.max(np.abs(out[inner] - lap[inner])) / np.max(np.abs(lap[inner]))
    assert err < 1e-9
    # degree 14 is NOT exact (the stencil is 12th order, not more)
    f14 = np.broadcast_to(x ** 14 + 0 * y + 0 * z, (n[2], n[1], n[0]))
    out14 = H.laplacian(np.ascontiguousarray(f14).ravel())[:, 0].reshape(n[2], n[1], n[0])
    lap14 = np.broadcast_to(182 * x ** 12 + 0 * y + 0 * z, (n[2], n[1], n[0]))
    assert np.max(np.abs(out14[inner] - lap14[inner])) > 1e-9 * np.max(np.abs(lap14[inner]))


# ----------------------------------------------------------------------------- P4
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_P4_dirichlet_equals_restricted_padded_periodic(axis):
    n, h = [14, 13, 15], (0.5, 0.45, 0.4)
    bc = [0, 0, 0]
    bc[axis] = 1
    wl_d = empty_atoms_workload(tuple(n), h, tuple(bc))
    npad = list(n)
    npad[axis] += 6
    wl_p = empty_atoms_workload(tuple(npad), h, (0, 0, 0))
    psi = rand((n[2], n[1], n[0]), 7)
    padded = np.zeros((npad[2], npad[1], npad[0]))
    padded[: n[2], : n[1], : n[0]] = psi
    out_d = orc.Hamiltonian(wl_d).laplacian(psi.ravel())[:, 0].reshape(n[2], n[1], n[0])
    out_p = orc.Hamiltonian(wl_p).laplacian(padded.ravel())[:, 0].reshape(npad[2], npad[1], npad[0])
    assert np.max(np.abs(out_d - out_p[: n[2], : n[1], : n[0]])) < 1e-12 * np.max(np.abs(out_d))


# ----------------------------------------------------------------------------- P5
def dense_H(wl, gw):
    """Dense H built entry by entry from the definition (readings R1, R2, R6-R9)."""
    nx, ny, nz = wl.n
    nd = wl.nd
    Hd = np.zeros((nd, nd))
    nn = (nx, ny, nz)
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                i = x + nx * (y + ny * z)
                c = (x, y, z)
                for ax in range(3):
                    for p in range(-6, 7):
                        q = c[ax] + p
                        if wl.bc[ax] == 0:
                            q %= nn[ax]
                        elif q < 0 or q >= nn[ax]:
                            continue
                        cc = list(c)
                        cc[ax] = q
                        j = cc[0] + nx * (cc[1] + ny * cc[2])
                        Hd[i, j] += -0.5 * gw[abs(p)] / wl.h[ax] ** 2
                Hd[i, i] += wl.veff[i]
    g0 = 0
    for J in range(wl.n_atoms):
        P = int(wl.n_proj[J])
        idx = wl.supp_idx[wl.supp_ptr[J]:wl.supp_ptr[J + 1]].astype(np.int64)
        tab = wl.chi[wl.chi_ptr[J]:wl.chi_ptr[J + 1]].reshape((idx.size, P), order="F")
        for q in range(P):
            Hd[np.ix_(idx, idx)] += wl.gamma[g0 + q] * np.outer(tab[:, q], tab[:, q])
        g0 += P
    return Hd


@pytest.fixture(scope="module")
def tiny_mixed(golden_dir):
    """13x14x16 anisotropic grid, bc = (P, P, D), two atoms, one straddling a periodic face and one
    cut by the Dirichlet face (pin P5)."""
    n, h = (13, 14, 16), (0.5, 0.45, 0.4)
    pos = np.array([[0.2, 3.1, 3.3], [4.1, 6.2, 0.7]])
    wl = wlmod.make_custom("tiny_mixed", n, h, (0, 0, 1), ns=5, degree=7, atom_pos=pos,
                           n_proj=[4, 9], rc=2.5, seed=11)
    gw = [float(x) for x in golden_weights(golden_dir)]
    Hd = dense_H(wl, gw)
    return wl, Hd


def test_P5_dense_brute_force_apply(tiny_mixed):
    wl, Hd = tiny_mixed
    assert np.max(np.abs(Hd - Hd.T)) < 1e-12
    X = rand((wl.nd, 5), 3)
    Y = orc.Hamiltonian(wl).apply(X)
    ref = Hd @ X
    assert np.max(np.abs(Y - ref)) / np.max(np.abs(ref)) < 1e-13
    # the pieces separately
    Hloc = orc.Hamiltonian(wl, nonlocal_on=False)
    Vnl = orc.Hamiltonian(wl).vnl_apply(X)
    assert np.max(np.abs(Hloc.apply(X) + Vnl - ref)) / np.max(np.abs(ref)) < 1e-13
    assert np.max(np.abs(Vnl)) > 1e-3        # the nonlocal term is really there


def test_P5_filter_equals_spectral_function(tiny_mixed):
    wl, Hd = tiny_mixed
    lam, V = np.linalg.eigh(Hd)
    assert lam[-1] <= wl.b + 1e-9 and lam[0] >= wl.a0 - 5.0
    X = rand((wl.nd, 3), 5)
    e, c = 0.5 * (wl.b - wl.a), 0.5 * (wl.b + wl.a)
    t0 = (wl.a0 - c) / e
    H = orc.Hamiltonian(wl)
    for m in (1, 2, 7, 12):
        Y = H.chebyshev_filter(X, m, wl.a, wl.b, wl.a0)
        ref = V @ ((cheb_T(m, (lam - c) / e) / cheb_T(m, np.array([t0]))[0])[:, None] * (V.T @ X))
        err = np.max(np.abs(Y - ref), axis=0) / np.linalg.norm(ref, axis=0)
        assert err.max() < 1e-11, (m, err)
    assert np.array_equal(H.chebyshev_filter(X, 0, wl.a, wl.b, wl.a0), X)
    with pytest.raises(ValueError):
        H.chebyshev_filter(X, 3, wl.b, wl.a, wl.a0)       # a >= b
    with pytest.raises(ValueError):
        H.chebyshev_filter(X, -1, wl.a, wl.b, wl.a0)


def test_P10_eigenvector_projection_is_diagonal(tiny_mixed):
    wl, Hd = tiny_mixed
    lam, V = np.linalg.eigh(Hd)
    Psi = np.asfortranarray(V[:, :6])
    Hs, Ms = orc.Hamiltonian(wl).project(Psi)
    assert np.max(np.abs(Ms - np.eye(6))) < 1e-12
    assert np.max(np.abs(Hs - np.diag(lam[:6]))) < 1e-11 * max(1.0, np.abs(lam).max())


# ----------------------------------------------------------------------------- P6
@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (1, 1, 0), (1, 0, 1),
                                (0, 1, 1), (1, 1, 1)])
@pytest.mark.parametrize("nonlocal_on", [False, True])
def test_P6_symmetry(bc, nonlocal_on):
    n, h = (13, 14, 15), (0.5, 0.45, 0.4)
    pos = np.array([[0.3, 2.9, 3.2], [5.9, 0.1, 5.5]])
    wl = wlmod.make_custom("sym", n, h, bc, 2, 4, pos, [9, 4], 2.5, seed=5)
    H = orc.Hamiltonian(wl, nonlocal_on=nonlocal_on)
    x, y = rand((wl.nd, 1), 1), rand((wl.nd, 1), 2)
    Hx, Hy = H.apply(x), H.apply(y)
    lhs, rhs = float(np.vdot(x, Hy)), float(np.vdot(Hx, y))
    assert abs(lhs - rhs) < 1e-12 * np.linalg.norm(x) * np.linalg.norm(Hy)


# ----------------------------------------------------------------------------- P7
def test_P7_plane_wave_Tm_scaling(golden_dir):
    """V_nl = 0, Veff = V0: plane waves are eigenvectors with lambda = -1/2 symbol + V0 and the
    filter multiplies them by T_m((lambda - c)/e) / T_m(t0)."""
    gw = [float(x) for x in golden_weights(golden_dir)]
    n, h = (24, 24, 24), (0.5, 0.5, 0.5)
    V0 = -0.7
    wl = empty_atoms_workload(n, h, (0, 0, 0), veff_kind=f"const:{V0}")
    H = orc.Hamiltonian(wl)
    a0, b = V0 - 0.1, 0.5 * 3 * (367616.0 / 51975.0) / 0.25 + V0 + 0.1
    a = a0 + 0.3 * (b - a0)
    e, c = 0.5 * (b - a), 0.5 * (b + a)
    t0 = (a0 - c) / e
    cols, lams = [], []
    g = np.arange(24) * 0.5
    for modes in [(0, 0, 0), (1, 0, 2), (3, 5, 7), (12, 12, 12), (11, 2, 0)]:
        k = [2 * math.pi * mm / 12.0 for mm in modes]
        cols.append(np.cos(k[0] * g[None, None, :] + k[1] * g[None, :, None] + k[2] * g[:, None, None]
                           + 0.4).ravel())
        sym = sum((gw[0] + 2 * sum(gw[p] * math.cos(p * k[ax] * 0.5) for p in range(1, 7))) / 0.25
                  for ax in range(3))
        lams.append(-0.5 * sym + V0)
    X = np.asfortranarray(np.stack(cols, axis=1))
    for m in (1, 10, 24):
        Y = H.chebyshev_filter(X, m, a, b, a0)
        for j, lam in enumerate(lams):
            fac = cheb_T(m, np.array([(lam - c) / e]))[0] / cheb_T(m, np.array([t0]))[0]
            assert np.max(np.abs(Y[:, j] - fac * X[:, j])) < 1e-12 * np.linalg.norm(X[:, j])
    # T_24(t0) is large (R3): the scaled form is what keeps this representable
    assert abs(cheb_T(24, np.array([t0]))[0]) > 1e9


def test_P7_single_atom_orthogonal_projectors():
    """One atom ON a grid point, equal h, support clear of faces: s, p, d projectors are exactly
    orthogonal on the grid, so V_nl chi_q = gamma_q ||chi_q||^2 chi_q (pin P7 (ii))."""
    n, h = (24, 24, 24), (0.4, 0.4, 0.4)
    pos = np.array([[12 * 0.4, 11 * 0.4, 13 * 0.4]])
    gamma = np.array([0.7, -0.3, 0.9, 0.2, -0.8, 0.5, 0.35, -0.45, 0.6])
    wl = wlmod.make_custom("one", n, h, (1, 1, 1), 1, 1, pos, [9], 3.0, gamma=gamma, veff_kind="zero")
    H = orc.Hamiltonian(wl)
    idx = wl.supp_idx.astype(np.int64)
    tab = wl.chi.reshape((idx.size, 9), order="F")
    G = tab.T @ tab
    assert np.max(np.abs(G - np.diag(np.diag(G)))) < 1e-12       # premise: orthogonal on the grid
    for q in range(9):
        v = np.zeros(wl.nd)
        v[idx] = tab[:, q]
        out = H.vnl_apply(v)[:, 0]
        ref = gamma[q] * G[q, q] * v
        assert np.max(np.abs(out - ref)) < 1e-12 * np.linalg.norm(ref)


# ----------------------------------------------------------------------------- P8
def test_P8_small_degrees_and_unscaled_recurrence():
    wl = wlmod.make_workload(0)
    H = orc.Hamiltonian(wl)
    X = wl.psi_columns([0, 7])
    a0, a, b = wl.a0, wl.a, wl.b
    e, c = 0.5 * (b - a), 0.5 * (b + a)
    HX = H.apply(X)
    Y1 = H.chebyshev_filter(X, 1, a, b, a0)
    ref1 = (HX - c * X) / (a0 - c)
    assert np.max(np.abs(Y1 - ref1)) < 1e-13 * np.linalg.norm(ref1)
    s1 = e / (a0 - c)
    s2 = 1.0 / (2.0 / s1 - s1)
    ref2 = (2 * s2 / e) * (H.apply(ref1) - c * ref1) - s1 * s2 * X
    Y2 = H.chebyshev_filter(X, 2, a, b, a0)
    assert np.max(np.abs(Y2 - ref2)) < 1e-13 * np.linalg.norm(ref2)
    # scaled * T_m(t0) == unscaled three-term recurrence T_{k+1} = 2 t T_k - T_{k-1}
    t0 = (a0 - c) / e
    Tprev, Tcur = X, (HX - c * X) / e
    for m in range(2, 6):
        Tnext = 2.0 * (H.apply(Tcur) - c * Tcur) / e - Tprev
        Tprev, Tcur = Tcur, Tnext
        Ym = H.chebyshev_filter(X, m, a, b, a0)
        Tm0 = cheb_T(m, np.array([t0]))[0]
        assert np.max(np.abs(Ym * Tm0 - Tcur)) < 1e-11 * np.max(np.abs(Tcur))


# ----------------------------------------------------------------------------- P9
def test_P9_column_independence():
    wl = wlmod.make_workload(0)
    H = orc.Hamiltonian(wl)
    X = wl.psi_columns(range(6))
    Y = H.chebyshev_filter(X, 4, wl.a, wl.b, wl.a0)
    Ysub = H.chebyshev_filter(X[:, [4, 1]], 4, wl.a, wl.b, wl.a0)
    assert np.array_equal(Y[:, [4, 1]], Ysub)


# ----------------------------------------------------------------------------- P10
def test_P10_gram_and_rotation_invariants():
    rng = np.random.default_rng(0)
    nd, ns = 1500, 12
    A = np.asfortranarray(rng.uniform(-1, 1, (nd, ns)))
    Qo, _ = np.linalg.qr(A)
    Ms = orc.gram(Qo, Qo)
    assert np.max(np.abs(Ms - np.eye(ns))) < 1e-13                  # orthonormal -> identity
    M = orc.gram(A, A)
    assert abs(np.trace(M) - np.linalg.norm(A) ** 2) < 1e-11 * np.linalg.norm(A) ** 2
    assert np.max(np.abs(M - M.T)) < 1e-13 * np.abs(M).max()
    assert np.linalg.eigvalsh(M).min() > 0                           # SPD
    B = np.asfortranarray(rng.uniform(-1, 1, (nd, ns)))
    G = orc.gram(A, B)
    assert np.max(np.abs(G - A.T @ B)) < 1e-12 * np.abs(G).max()     # textbook product
    I, J = [3, 0, 11], [5, 5, 2, 9]
    assert np.array_equal(orc.gram(A, B, I, J), G[np.ix_(I, J)])     # sampled entries = same sums
    Q, _ = np.linalg.qr(rng.normal(size=(ns, ns)))
    R = orc.rotate(A, Q)
    assert np.max(np.abs(R - A @ Q)) < 1e-13 * np.abs(R).max()
    assert abs(np.linalg.norm(R) - np.linalg.norm(A)) < 1e-12 * np.linalg.norm(A)
    back = orc.rotate(R, np.asfortranarray(Q.T))
    assert np.max(np.abs(back - A)) < 1e-13
    rows = [0, 17, 1499, 3]
    assert np.array_equal(orc.rotate(A, Q, rows), R[rows, :])
    # a non-symmetric Q distinguishes Psi Q from Psi Q^T
    assert np.max(np.abs(R - A @ Q.T)) > 1e-3


def test_P10_project_of_rotated_block():
    wl = wlmod.make_workload(0)
    H = orc.Hamiltonian(wl)
    Psi = wl.psi_columns(range(8))
    Q, _ = np.linalg.qr(np.random.default_rng(3).normal(size=(8, 8)))
    Hs, Ms = H.project(Psi)
    Hs2, Ms2 = H.project(orc.rotate(Psi, Q))
    assert np.linalg.norm(Hs2 - Q.T @ Hs @ Q) < 1e-12 * np.linalg.norm(Hs)
    assert np.linalg.norm(Ms2 - Q.T @ Ms @ Q) < 1e-12 * np.linalg.norm(Ms)
    assert np.linalg.norm(Hs - Hs.T) < 1e-12 * np.linalg.norm(Hs)


def test_f64_build_agrees_with_long_double_build():
    """The plain-FP64 build (timed as cpu_baseline) is the same program with acc_t = double."""
    wl = wlmod.make_workload(0)
    X = wl.psi_columns([1, 2])
    Yl = orc.Hamiltonian(wl, acc="ld").chebyshev_filter(X, wl.degree, wl.a, wl.b, wl.a0)
    Yd = orc.Hamiltonian(wl, acc="f64").chebyshev_filter(X, wl.degree, wl.a, wl.b, wl.a0)
    err = np.max(np.abs(Yl - Yd), axis=0) / np.linalg.norm(Yl, axis=0)
    assert err.max() < 1e-13
    assert orc._lib("ld").oracle_acc_bits() >= 80 and orc._lib("f64").oracle_acc_bits() == 64
