"""Pins of oracle/chefsi_next_oracle.c, CPU only.  Each oracle function is checked against
something other than itself: exact rationals, closed forms, invariants, brute force written independently here in numpy,
or a LAPACK routine on the special case it reduces to.

  N1  first-derivative weights: exact rationals (tests/golden/fd1_weights_r6.txt), odd-moment conditions, textbook radii
  N2  gradient on plane waves: symbol  sum_p 2 w_p sin(p k h) / h  (closed form), anisotropic grid, every axis
  N3  gradient: polynomial exactness to degree 12, antisymmetry <x, D y> = -<D x, y> on periodic axes, Dirichlet =
      restricted zero-padded periodic
  N4  chi^T X and the nonlocal force against a dense brute force built entry by entry; force = -dE_nl/dR by finite
      differences of the energy on a rigidly shifted projector (Gaussian s projector, closed form)
  N5  generalized eigenproblem: residual, M-orthonormality, ascending order, diagonal closed form, 2 x 2 closed form,
      LAPACK eigenvalues (scipy.linalg.eigh), degenerate spectrum, not-positive-definite error
  N6  complex operator: Hermiticity, theta = 0 equals the real operator, Bloch plane waves (closed-form eigenvalue),
      dense brute-force H(k) with projector images across a periodic face, filter = polynomial of H(k), Gram / rotation
      against numpy
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2302_09708_b200 import workloads as wlmod

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ---------------------------------------------------------------------------------------------------------------------
# N1
def test_fd1_weights_exact_rationals_and_moments(golden_dir):
    gold = {}
    for ln in open(os.path.join(golden_dir, "fd1_weights_r6.txt")):
        ln = ln.split("#")[0].strip()
        if ln:
            p, frac = ln.split()
            gold[int(p)] = Fraction(frac)
    w = orc.fd1_weights(6)
    assert w[0] == 0.0
    for p in range(1, 7):
        assert abs(w[p] - float(gold[p])) <= 1e-17 * max(1.0, abs(float(gold[p]))) + 1e-19
    # exact moment conditions on the rationals: sum_p 2 w_p p = 1, sum_p 2 w_p p^(2j+1) = 0 for j = 1..5, != 0 for j = 6
    assert sum(2 * gold[p] * p for p in gold) == 1
    for j in range(1, 6):
        assert sum(2 * gold[p] * p ** (2 * j + 1) for p in gold) == 0
    assert sum(2 * gold[p] * p ** 13 for p in gold) != 0
    # textbook radii
    assert np.allclose(orc.fd1_weights(1)[1:], [0.5], rtol=0, atol=1e-17)
    assert np.allclose(orc.fd1_weights(2)[1:], [2.0 / 3.0, -1.0 / 12.0], rtol=0, atol=1e-17)
    assert np.allclose(orc.fd1_weights(3)[1:], [0.75, -0.15, 1.0 / 60.0], rtol=0, atol=1e-17)


def _grid_wl(n, h, bc, atoms=None, projs=None, rc=2.0, seed=3, ns=3, gamma=None):
    pos = np.zeros((0, 3)) if atoms is None else np.asarray(atoms, float)
    return wlmod.make_custom("g", n, h, bc, ns, 4, pos, [] if projs is None else projs, rc, seed=seed, gamma=gamma)


# ---------------------------------------------------------------------------------------------------------------------
# N2
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_gradient_plane_wave_symbol(axis):
    n, h = (16, 18, 20), (0.5, 0.45, 0.4)
    wl = _grid_wl(n, h, (0, 0, 0))
    F = orc.Forces(wl)
    w = [Fraction(6, 7), Fraction(-15, 56), Fraction(5, 63), Fraction(-1, 56), Fraction(1, 385), Fraction(-1, 5544)]
    x = np.arange(n[0])[:, None, None] * h[0]
    y = np.arange(n[1])[None, :, None] * h[1]
    z = np.arange(n[2])[None, None, :] * h[2]
    for m in [(1, 0, 0), (2, 3, 1), (0, 5, 2), (7, 1, 4)]:
        k = [2 * math.pi * m[a] / (n[a] * h[a]) for a in range(3)]
        phase = k[0] * x + k[1] * y + k[2] * z + 0.3
        psi = np.sin(phase).ravel(order="F")
        sym = sum(2 * float(w[p - 1]) * math.sin(p * k[axis] * h[axis]) for p in range(1, 7)) / h[axis]
        exact = (sym * np.cos(phase)).ravel(order="F")
        got = F.gradient(psi, axis)[:, 0]
        assert np.max(np.abs(got - exact)) <= 1e-13 * max(1.0, abs(sym))
        # and the symbol approximates k to 12th order (spot value: k h = 0.5 -> relative error ~ 1e-7 or better)
        if abs(k[axis]) > 0 and abs(k[axis] * h[axis]) < 0.6:
            assert abs(sym / k[axis] - 1.0) < 1e-6


# ---------------------------------------------------------------------------------------------------------------------
# N3
def test_gradient_polynomial_exactness_and_dirichlet_and_antisymmetry():
    n, h = (15, 14, 16), (0.5, 0.45, 0.4)
    wl = _grid_wl(n, h, (1, 1, 1))
    F = orc.Forces(wl)
    X, Y, Z = np.meshgrid(np.arange(n[0]) * h[0], np.arange(n[1]) * h[1], np.arange(n[2]) * h[2], indexing="ij")
    X, Y, Z = X - 3.1, Y - 2.7, Z - 3.3          # centred coordinates keep the monomials O(1)
    inner = np.zeros(n, bool)
    inner[6:-6, 6:-6, 6:-6] = True
    for (a, b, c) in [(12, 0, 0), (0, 12, 0), (0, 0, 12), (5, 4, 3), (1, 0, 11), (3, 9, 0)]:
        f = X ** a * Y ** b * Z ** c
        exact = [a * X ** max(a - 1, 0) * Y ** b * Z ** c if a else 0 * X,
                 b * X ** a * Y ** max(b - 1, 0) * Z ** c if b else 0 * X,
                 c * X ** a * Y ** b * Z ** max(c - 1, 0) if c else 0 * X]
        for axis in range(3):
            got = F.gradient(f.ravel(order="F"), axis)[:, 0].reshape(n, order="F")
            scale = max(1.0, np.max(np.abs(exact[axis][inner])))
            assert np.max(np.abs(got[inner] - exact[axis][inner])) <= 2e-10 * scale
    # degree 13 is NOT exact (the order is 12)
    f = X ** 13
    got = F.gradient(f.ravel(order="F"), 0)[:, 0].reshape(n, order="F")
    assert np.max(np.abs(got[inner] - (13 * X ** 12)[inner])) > 1e-8
    # Dirichlet(n) = restriction of Periodic(n + 6) applied to the zero-padded field, axis by axis
    rng = np.random.default_rng(0)
    for axis in range(3):
        bc = [0, 0, 0]
        bc[axis] = 1
        wl_d = _grid_wl(n, h, tuple(bc))
        npad = list(n)
        npad[axis] += 6
        wl_p = _grid_wl(tuple(npad), h, (0, 0, 0))
        f = rng.normal(size=n)
        fp = np.zeros(npad)
        sl = [slice(None)] * 3
        sl[axis] = slice(0, n[axis])
        fp[tuple(sl)] = f
        gd = orc.Forces(wl_d).gradient(f.ravel(order="F"), axis)[:, 0].reshape(n, order="F")
        gp = orc.Forces(wl_p).gradient(fp.ravel(order="F"), axis)[:, 0].reshape(npad, order="F")
        assert np.max(np.abs(gd - gp[tuple(sl)])) <= 1e-14 * np.max(np.abs(gd))
    # antisymmetry on periodic axes, and its failure mode: <x, D y> + <D x, y> = 0
    wl_p = _grid_wl(n, h, (0, 0, 0))
    Fp = orc.Forces(wl_p)
    x, y = rng.normal(size=wl_p.nd), rng.normal(size=wl_p.nd)
    for axis in range(3):
        s = x @ Fp.gradient(y, axis)[:, 0] + Fp.gradient(x, axis)[:, 0] @ y
        assert abs(s) <= 1e-11 * np.linalg.norm(x) * np.linalg.norm(y)


# ---------------------------------------------------------------------------------------------------------------------
# N4
def _dense_gradient(n, h, bc, axis, w):
    nx, ny, nz = n
    nd = nx * ny * nz
    D = np.zeros((nd, nd))
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                i = x + nx * (y + ny * z)
                c = [x, y, z]
                for p in range(1, len(w) + 1):
                    for sg in (-1, 1):
                        q = c[axis] + sg * p
                        if bc[axis] == 0:
                            q %= n[axis]
                        elif q < 0 or q >= n[axis]:
                            continue
                        cc = list(c)
                        cc[axis] = q
                        D[i, cc[0] + nx * (cc[1] + ny * cc[2])] += sg * w[p - 1] / h[axis]
    return D


def test_projection_and_force_dense_brute_force():
    n, h, bc = (13, 14, 15), (0.5, 0.45, 0.4), (0, 0, 1)
    pos = np.array([[0.3, 3.0, 3.1], [4.0, 0.2, 5.5]])       # supports straddle periodic faces and a Dirichlet face
    wl = wlmod.make_custom("force", n, h, bc, 5, 4, pos, [4, 9], 2.2, seed=13)
    F = orc.Forces(wl)
    X = wl.psi_columns(range(wl.ns))
    occ = wl.occupations()
    w = [6 / 7, -15 / 56, 5 / 63, -1 / 56, 1 / 385, -1 / 5544]
    # chi^T X, row by row, from the tables
    Wd = np.zeros((int(wl.n_proj.sum()), wl.ns))
    po = 0
    for J in range(wl.n_atoms):
        idx = wl.supp_idx[wl.supp_ptr[J]:wl.supp_ptr[J + 1]]
        tab = wl.chi[wl.chi_ptr[J]:wl.chi_ptr[J + 1]].reshape((len(idx), wl.n_proj[J]), order="F")
        Wd[po:po + wl.n_proj[J]] = tab.T @ X[idx]
        po += wl.n_proj[J]
    assert np.max(np.abs(F.nl_project(X) - Wd)) <= 1e-13 * np.max(np.abs(Wd))
    Fd = np.zeros((wl.n_atoms, 3))
    for a in range(3):
        D = _dense_gradient(n, h, bc, a, w)
        DX = D @ X
        assert np.max(np.abs(F.gradient(X, a) - DX)) <= 1e-13 * np.max(np.abs(DX))
        po = 0
        for J in range(wl.n_atoms):
            idx = wl.supp_idx[wl.supp_ptr[J]:wl.supp_ptr[J + 1]]
            tab = wl.chi[wl.chi_ptr[J]:wl.chi_ptr[J + 1]].reshape((len(idx), wl.n_proj[J]), order="F")
            G = tab.T @ DX[idx]
            gam = wl.gamma[po:po + wl.n_proj[J]]
            Fd[J, a] = -2.0 * np.sum(occ[None, :] * gam[:, None] * Wd[po:po + wl.n_proj[J]] * G)
            po += wl.n_proj[J]
    got = F.nonlocal_force(X, occ)
    assert np.max(np.abs(got - Fd)) <= 1e-12 * np.max(np.abs(Fd))


def test_force_is_minus_energy_derivative():
    """F = -dE_nl/dR: smooth orbitals, one s projector chi(r) = exp(-|r - R|^2 / 2) sampled on a fine periodic grid with a
    support that covers the whole Gaussian; E_nl(R) = sum_n g_n gamma (chi_R^T psi_n)^2 from the tables at R +- d, central
    difference in R against the oracle's force.  (The oracle applies the gradient to the ORBITALS; the energy moves the
    PROJECTOR: the two agree up to the 12th-order stencil error and the truncation of the Gaussian.)"""
    n, hh = (30, 30, 30), 0.35
    L = n[0] * hh
    gamma = np.array([0.8])
    x = np.arange(n[0]) * hh
    Xg, Yg, Zg = np.meshgrid(x, x, x, indexing="ij")
    k = 2 * math.pi / L
    psi = np.stack([(np.sin(k * Xg + 0.2) * np.cos(2 * k * Yg) + 0.3 * np.cos(k * Zg)).ravel(order="F"),
                    (np.cos(2 * k * Xg - 0.4) + np.sin(k * Yg + k * Zg)).ravel(order="F")], axis=1)
    occ = np.array([2.0, 1.3])

    def energy(R):
        wl = wlmod.make_custom("e", n, (hh,) * 3, (0, 0, 0), 2, 1, np.array([R]), [1], 5.2, gamma=gamma)
        W = orc.Forces(wl).nl_project(psi)
        return float(np.sum(occ * gamma[0] * W[0] ** 2)), wl

    R0 = np.array([4.1, 4.3, 3.9])
    _, wl0 = energy(R0)
    Fo = orc.Forces(wl0).nonlocal_force(psi, occ)[0]
    d = 1e-3
    for a in range(3):
        e = np.zeros(3)
        e[a] = d
        Ep, _ = energy(R0 + e)
        Em, _ = energy(R0 - e)
        fd = -(Ep - Em) / (2 * d)
        assert abs(fd - Fo[a]) <= 1e-4 * max(1.0, abs(Fo).max()), (a, fd, Fo[a])


# ---------------------------------------------------------------------------------------------------------------------
# N5
def _rand_pencil(n, rng, cond=1e3):
    A = rng.normal(size=(n, n))
    H = A + A.T
    Q, _ = np.linalg.qr(rng.normal(size=(n, n)))
    M = Q @ np.diag(np.geomspace(1.0, cond, n)) @ Q.T
    return np.asfortranarray(H), np.asfortranarray((M + M.T) / 2)


@pytest.mark.parametrize("n", [1, 2, 5, 32, 97])
def test_sygv_residual_orthonormality_order_and_lapack(n):
    import scipy.linalg as sl
    rng = np.random.default_rng(100 + n)
    H, M = _rand_pencil(n, rng)
    D, Z = orc.sygv(H, M)
    assert np.all(np.diff(D) >= 0)
    scale = np.linalg.norm(H) + np.linalg.norm(M) * np.abs(D).max()
    assert np.linalg.norm(H @ Z - M @ Z * D[None, :]) <= 1e-13 * scale * np.linalg.norm(Z)
    assert np.max(np.abs(Z.T @ M @ Z - np.eye(n))) <= 1e-12
    ref = sl.eigh(H, M, eigvals_only=True)                    # LAPACK dsygvd on the same pencil
    assert np.max(np.abs(D - ref)) <= 1e-12 * max(1.0, np.abs(ref).max())


def test_sygv_closed_forms_and_errors():
    # diagonal pencil: eigenvalues a_i / b_i, eigenvectors e_i / sqrt(b_i)
    a = np.array([3.0, -1.0, 0.5, 2.0])
    b = np.array([2.0, 4.0, 0.25, 1.0])
    D, Z = orc.sygv(np.diag(a), np.diag(b))
    lam = a / b
    order = np.argsort(lam, kind="stable")
    assert np.allclose(D, lam[order], rtol=0, atol=1e-15)
    for c, i in enumerate(order):
        e = np.zeros(4)
        e[i] = 1.0 / math.sqrt(b[i])
        assert np.allclose(np.abs(Z[:, c]), e, rtol=0, atol=1e-15)
    # 2 x 2 with M = I: lambda = (a + d)/2 -+ sqrt(((a - d)/2)^2 + c^2)
    H = np.array([[2.0, 0.7], [0.7, -1.0]])
    D, Z = orc.sygv(H, np.eye(2))
    r = math.hypot(1.5, 0.7)
    assert np.allclose(D, [0.5 - r, 0.5 + r], rtol=0, atol=1e-15)
    # degenerate spectrum: H = M gives D = 1 (n-fold) and any M-orthonormal Z
    rng = np.random.default_rng(7)
    _, M = _rand_pencil(6, rng)
    D, Z = orc.sygv(M, M)
    assert np.allclose(D, 1.0, rtol=0, atol=1e-13) and np.max(np.abs(Z.T @ M @ Z - np.eye(6))) <= 1e-12
    with pytest.raises(ValueError):
        orc.sygv(np.eye(3), np.diag([1.0, -1.0, 1.0]))         # Ms not positive definite


def test_sygv_on_a_chefsi_subspace():
    """The pencil the method produces: Hs = X^T H X, Ms = X^T X of filtered orbitals; rotating with Z
    gives M-orthonormal Ritz vectors whose Rayleigh quotients are D."""
    wl = wlmod.make_workload(0)
    H = orc.Hamiltonian(wl)
    X = H.chebyshev_filter(wl.psi_columns(range(12)), 6, wl.a, wl.b, wl.a0)
    Hs, Ms = H.project(X)
    D, Z = orc.sygv(Hs, Ms)
    R = orc.rotate(X, Z)
    Hs2, Ms2 = H.project(R)
    assert np.max(np.abs(Ms2 - np.eye(12))) <= 1e-10
    assert np.max(np.abs(Hs2 - np.diag(D))) <= 1e-10 * max(1.0, np.abs(D).max())


# ---------------------------------------------------------------------------------------------------------------------
# N6
def _dense_hk(wl, theta):
    """H(k) entry by entry from the definition (independent of the oracle's loops)."""
    nx, ny, nz = wl.n
    nd = wl.nd
    r = wl.fd_order // 2
    w2 = {0: Fraction(-5369, 1800), 1: Fraction(12, 7), 2: Fraction(-15, 56), 3: Fraction(10, 189), 4: Fraction(-1, 112),
          5: Fraction(2, 1925), 6: Fraction(-1, 16632)}
    assert r == 6
    Hd = np.zeros((nd, nd), dtype=complex)
    n = (nx, ny, nz)
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                i = x + nx * (y + ny * z)
                c = (x, y, z)
                Hd[i, i] += wl.veff[i]
                for a in range(3):
                    for p in range(-r, r + 1):
                        q = c[a] + p
                        ph = 1.0
                        if wl.bc[a] == 0:
                            wraps = q // n[a]
                            q -= wraps * n[a]
                            ph = np.exp(1j * wraps * theta[a])
                        elif q < 0 or q >= n[a]:
                            continue
                        cc = list(c)
                        cc[a] = q
                        Hd[i, cc[0] + nx * (cc[1] + ny * cc[2])] += -0.5 * float(w2[abs(p)]) / wl.h[a] ** 2 * ph
    po = 0
    for J in range(wl.n_atoms):
        s0, s1 = wl.supp_ptr[J], wl.supp_ptr[J + 1]
        idx = wl.supp_idx[s0:s1]
        tab = wl.chi[wl.chi_ptr[J]:wl.chi_ptr[J + 1]].reshape((s1 - s0, wl.n_proj[J]), order="F")
        phi = wl.supp_shift[s0:s1].astype(float) @ np.where(np.asarray(wl.bc) == 0, theta, 0.0)
        ct = tab * np.exp(-1j * phi)[:, None]                 # chi~ = chi exp(-i phi)
        Hd[np.ix_(idx, idx)] += (ct * wl.gamma[po:po + wl.n_proj[J]][None, :]) @ ct.conj().T
        po += wl.n_proj[J]
    return Hd


def test_hk_dense_brute_force_hermiticity_and_filter():
    pos = np.array([[0.2, 3.1, 3.0], [3.6, 0.3, 0.4]])       # supports cross periodic faces: image shifts +-1 present
    wl = wlmod.make_custom("hk", (13, 14, 13), (0.5, 0.45, 0.4), (0, 0, 1), 3, 5, pos, [4, 9], 2.3, seed=19)
    assert set(np.unique(wl.supp_shift)) >= {-1, 0, 1} or set(np.unique(wl.supp_shift)) >= {-1, 0}
    theta = np.array([0.7, -1.9, 0.4])
    Hk = orc.HamiltonianK(wl, theta)
    Hd = _dense_hk(wl, theta)
    assert np.max(np.abs(Hd - Hd.conj().T)) <= 1e-13 * np.max(np.abs(Hd))          # Hermitian by construction
    X = wl.psi_columns_complex(range(wl.ns))
    Y = Hk.apply(X)
    ref = Hd @ X
    assert np.max(np.abs(Y - ref)) <= 1e-13 * np.max(np.abs(ref))
    # <x, H y> = conj(<y, H x>)
    x, y = X[:, 0], X[:, 1]
    assert abs(np.vdot(x, Y[:, 1]) - np.conj(np.vdot(y, Y[:, 0]))) <= 1e-11 * np.linalg.norm(x) * np.linalg.norm(Y[:, 1])
    # filter = V T_m((Lambda - c)/e) / T_m(t0) V^H X
    lam, V = np.linalg.eigh(Hd)
    a0, a, b = lam.min() - 0.5, lam.min() + 0.3 * (lam.max() - lam.min()), lam.max() + 0.1
    e, c = (b - a) / 2, (b + a) / 2

    def T(m, t):
        t = np.asarray(t, float)
        out = np.empty_like(t)
        ins = np.abs(t) <= 1
        out[ins] = np.cos(m * np.arccos(t[ins]))
        o = ~ins
        out[o] = np.sign(t[o]) ** m * np.cosh(m * np.arccosh(np.abs(t[o])))
        return out

    for m in (1, 2, 7):
        ref = V @ ((T(m, (lam - c) / e) / T(m, np.array([(a0 - c) / e]))[0])[:, None] * (V.conj().T @ X))
        got = Hk.chebyshev_filter(X, m, a, b, a0)
        assert np.max(np.abs(got - ref)) <= 1e-12 * np.max(np.abs(ref))


def test_hk_gamma_point_limit_and_bloch_plane_waves():
    pos = np.array([[1.0, 2.0, 3.0]])
    wl = wlmod.make_custom("hk0", (14, 13, 15), (0.5, 0.45, 0.4), (0, 1, 0), 3, 5, pos, [4], 2.0, seed=23)
    X = wl.psi_columns(range(3))
    Y0 = orc.HamiltonianK(wl, (0.0, 0.0, 0.0)).apply(X.astype(complex))
    Yr = orc.Hamiltonian(wl).apply(X)
    assert np.max(np.abs(Y0.imag)) == 0.0 and np.max(np.abs(Y0.real - Yr)) <= 1e-14 * np.max(np.abs(Yr))
    # Bloch plane wave on a fully periodic grid, Veff = V0, no atoms: psi = exp(i (G + k) r) obeys the boundary phase
    # theta_a = k_a L_a and is an eigenvector with lambda = -1/2 sum_a symbol_a((G + k)_a) + V0
    n, h = (14, 16, 13), (0.5, 0.45, 0.4)
    wlp = wlmod.make_custom("pw", n, h, (0, 0, 0), 1, 1, np.zeros((0, 3)), [], 2.0, veff_kind="const:0.37")
    w2 = [-5369 / 1800, 12 / 7, -15 / 56, 10 / 189, -1 / 112, 2 / 1925, -1 / 16632]
    theta = np.array([0.9, -0.5, 2.2])
    Lbox = [n[a] * h[a] for a in range(3)]
    kv = [theta[a] / Lbox[a] for a in range(3)]
    m = (2, -1, 3)
    q = [2 * math.pi * m[a] / Lbox[a] + kv[a] for a in range(3)]
    x = np.arange(n[0])[:, None, None] * h[0]
    y = np.arange(n[1])[None, :, None] * h[1]
    z = np.arange(n[2])[None, None, :] * h[2]
    psi = np.exp(1j * (q[0] * x + q[1] * y + q[2] * z)).ravel(order="F")
    lam = 0.37 - 0.5 * sum((w2[0] + 2 * sum(w2[p] * math.cos(p * q[a] * h[a]) for p in range(1, 7))) / h[a] ** 2
                           for a in range(3))
    Y = orc.HamiltonianK(wlp, theta).apply(psi)[:, 0]
    assert np.max(np.abs(Y - lam * psi)) <= 1e-12 * abs(lam)


def test_gram_k_and_rotate_k():
    rng = np.random.default_rng(5)
    A = rng.normal(size=(200, 7)) + 1j * rng.normal(size=(200, 7))
    B = rng.normal(size=(200, 5)) + 1j * rng.normal(size=(200, 5))
    G = orc.gram_k(A, B)
    assert np.max(np.abs(G - A.conj().T @ B)) <= 1e-13 * np.max(np.abs(G))
    M = orc.gram_k(A, A)
    assert np.max(np.abs(M - M.conj().T)) <= 1e-14 * np.max(np.abs(M)) and np.all(np.linalg.eigvalsh(M) > 0)
    Q = rng.normal(size=(7, 7)) + 1j * rng.normal(size=(7, 7))       # not Hermitian, not unitary: Q vs Q^T vs Q^H differ
    R = orc.rotate_k(A, Q)
    assert np.max(np.abs(R - A @ Q)) <= 1e-13 * np.max(np.abs(R))
