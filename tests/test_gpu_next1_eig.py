"""GPU parity: the generalized symmetric eigenproblem Hs Z = Ms Z D on the device
(sparc_gpu_eigensolve) against oracle/chefsi_next_oracle.c's oracle_sygv (E1-E4).  Several results are correct (sign of
each eigenvector, rotations inside degenerate eigenspaces): what is unique -- the eigenvalues -- is compared entry by entry,
and the rest is checked for validity: residual, M-orthonormality, ascending order, and the invariant subspaces agree with
the oracle's (|Z_o^T Ms Z| is a signed permutation-free identity for a non-degenerate spectrum)."""
import math
import time

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
def g(api):
    wl = wlmod.make_custom("eig_ctx", (14, 14, 14), (0.5,) * 3, (0, 0, 0), 2, 2, np.zeros((0, 3)), [], 2.0, seed=3)
    ctx = api.SparcGpu(wl)
    yield ctx
    ctx.close()


def rand_pencil(n, rng, cond=1e3):
    A = rng.normal(size=(n, n))
    H = A + A.T
    Q, _ = np.linalg.qr(rng.normal(size=(n, n)))
    M = Q @ np.diag(np.geomspace(1.0, cond, n)) @ Q.T
    return np.asfortranarray(H), np.asfortranarray((M + M.T) / 2)


def solve(torch, api, g, H, M):
    Hd = api.colmajor_from_numpy(H)
    Md = api.colmajor_from_numpy(M)
    D, Z, info = g.eigensolve(Hd, Md)
    torch.cuda.synchronize()
    assert np.array_equal(api.colmajor_to_numpy(Hd), H) and np.array_equal(api.colmajor_to_numpy(Md), M)   # inputs untouched
    return D.cpu().numpy(), api.colmajor_to_numpy(Z), info.cpu().numpy()


def check(H, M, D, Z, Do=None, tag=""):
    n = H.shape[0]
    assert np.all(np.diff(D) >= 0), "eigenvalues must ascend"
    scale = np.linalg.norm(H) + np.linalg.norm(M) * np.abs(D).max()
    res = np.linalg.norm(H @ Z - M @ Z * D[None, :]) / (scale * np.linalg.norm(Z))
    orth = np.max(np.abs(Z.T @ M @ Z - np.eye(n)))
    dev = None if Do is None else float(np.max(np.abs(D - Do)) / max(1.0, np.abs(Do).max()))
    print(f"[parity] eigensolve {tag} n={n}: residual {res:.2e}, |Z^T M Z - I| {orth:.2e}, |D - D_oracle| {dev}")
    assert res <= 1e-13
    assert orth <= 1e-11
    if Do is not None:
        assert dev <= 1e-11


@pytest.mark.parametrize("n", [1, 2, 3, 5, 32, 63, 64, 65, 97, 130, 257])
def test_eigensolve_against_oracle(torch, api, g, n):
    rng = np.random.default_rng(100 + n)
    H, M = rand_pencil(n, rng)
    D, Z, info = solve(torch, api, g, H, M)
    assert info[0] == 0, f"status {info[0]}"
    assert 1 <= info[1] <= 20 or n == 1
    Do, Zo = orc.sygv(H, M)
    check(H, M, D, Z, Do, "random pencil")
    if n > 1:      # non-degenerate spectrum: each device eigenvector is +- the oracle's
        S = np.abs(Zo.T @ M @ Z)
        assert np.max(np.abs(S - np.eye(n))) <= 1e-8


def test_eigensolve_closed_forms_and_degenerate(torch, api, g):
    a = np.array([3.0, -1.0, 0.5, 2.0])
    b = np.array([2.0, 4.0, 0.25, 1.0])
    D, Z, info = solve(torch, api, g, np.diag(a), np.diag(b))
    lam = a / b
    order = np.argsort(lam, kind="stable")
    assert info[0] == 0 and np.allclose(D, lam[order], rtol=0, atol=1e-14)
    for c, i in enumerate(order):
        e = np.zeros(4)
        e[i] = 1.0 / math.sqrt(b[i])
        assert np.allclose(np.abs(Z[:, c]), e, rtol=0, atol=1e-14)
    H = np.array([[2.0, 0.7], [0.7, -1.0]])
    D, Z, info = solve(torch, api, g, H, np.eye(2))
    r = math.hypot(1.5, 0.7)
    assert np.allclose(D, [0.5 - r, 0.5 + r], rtol=0, atol=1e-14)
    rng = np.random.default_rng(7)
    _, M = rand_pencil(6, rng)
    D, Z, info = solve(torch, api, g, M, M)                  # n-fold eigenvalue 1: any M-orthonormal Z is right
    assert info[0] == 0 and np.allclose(D, 1.0, rtol=0, atol=1e-13)
    check(M, M, D, Z, None, "H = M")
    D, Z, info = solve(torch, api, g, np.zeros((5, 5)), np.eye(5))    # H = 0
    assert info[0] == 0 and np.allclose(D, 0.0, atol=1e-15)
    # Ms not positive definite: status 1, no hang, no exception
    D, Z, info = solve(torch, api, g, np.eye(3), np.diag([1.0, -1.0, 1.0]))
    assert info[0] == 1


def test_chefsi_step_without_host_hop(torch, api):
    """filter -> project -> eigensolve -> rotate entirely on the device (Algorithm 1), configs[0]: the
    rotated orbitals are M-orthonormal Ritz vectors whose Rayleigh quotients are D, and D matches the oracle's for the
    oracle's own filtered block."""
    wl = wlmod.make_workload(0)
    gg = api.SparcGpu(wl)
    psi = torch.empty((wl.ns, wl.nd), dtype=torch.float64, device="cuda")
    api.fill_uniform(psi, wl.seed, wlmod.STREAM_PSI, 0, -1.0, 1.0)
    gg.chebyshev_filter(psi, wl.degree, wl.a, wl.b, wl.a0)
    Hs, Ms = gg.project(psi)
    D, Z, info = gg.eigensolve(Hs, Ms)
    gg.rotate(psi, Z)
    Hs2, Ms2 = gg.project(psi)
    torch.cuda.synchronize()
    assert info.cpu().numpy()[0] == 0
    Dn = D.cpu().numpy()
    assert np.max(np.abs(api.colmajor_to_numpy(Ms2) - np.eye(wl.ns))) <= 1e-9
    assert np.max(np.abs(api.colmajor_to_numpy(Hs2) - np.diag(Dn))) <= 1e-9 * max(1.0, np.abs(Dn).max())
    H = orc.Hamiltonian(wl)
    O = H.chebyshev_filter(wl.psi(), wl.degree, wl.a, wl.b, wl.a0)
    Hs_o, Ms_o = H.project(O)
    Do, _ = orc.sygv(Hs_o, Ms_o)
    # the filtered block is ill-conditioned (the filter amplifies the wanted end by orders of magnitude): eigenvalues of the
    # pencil are determined to ~cond(Ms) * eps
    cond = np.linalg.cond(Ms_o)
    print(f"[parity] cfg0 Ritz values: max |D - D_oracle| = {np.max(np.abs(Dn - Do)):.2e}, cond(Ms) = {cond:.1e}")
    assert np.max(np.abs(Dn - Do)) <= 1e-13 * cond * max(1.0, np.abs(Do).max())
    gg.close()


@pytest.mark.parametrize("n", [256, 1024, 2048, 4096])
def test_eigensolve_subspace_sizes(torch, api, g, n):
    """The subspace sizes of configs[1] (256), configs[2] (1024) and configs[3] (4096), and 2048 in between: validity checks
    (residual, M-orthonormality, ascending D) + LAPACK eigenvalues (the oracle's long double Jacobi takes minutes at 1024),
    with the device time.  configs[4]'s 7680 is beyond what the Jacobi solver does in useful time."""
    import scipy.linalg as sl
    rng = np.random.default_rng(n)
    H, M = rand_pencil(n, rng, cond=1e2)
    Hd, Md = api.colmajor_from_numpy(H), api.colmajor_from_numpy(M)
    g.eigensolve(Hd, Md)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    D, Z, info = g.eigensolve(Hd, Md)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    info = info.cpu().numpy()
    print(f"[time] eigensolve n={n}: {dt * 1e3:.1f} ms, {info[1]} sweeps")
    assert info[0] == 0
    ref = sl.eigh(H, M, eigvals_only=True)
    check(H, M, D.cpu().numpy(), api.colmajor_to_numpy(Z), ref, "vs LAPACK")


def test_eigensolve_argument_errors(torch, api, g):
    """n beyond the shared-memory limit of a column pair is UNSUPPORTED (-2), a short workspace is -5, n = 0 is a no-op."""
    import ctypes as C
    lib = g.lib
    one = torch.zeros(4, dtype=torch.float64, device="cuda")
    p = C.c_void_p(one.data_ptr())
    g._workspace(api.OP_EIGENSOLVE, 8, 0)
    assert lib.sparc_gpu_eigensolve(g._ctx, 0, p, p, p, p, None, p, None) == 0
    assert lib.sparc_gpu_eigensolve(g._ctx, 40000, p, p, p, p, None, p, None) == -2
    assert lib.sparc_gpu_eigensolve(g._ctx, 12801, p, p, p, p, None, p, None) == -2
    assert lib.sparc_gpu_eigensolve(g._ctx, -1, p, p, p, p, None, p, None) == -1
    declared = g._ws.numel()
    try:        # declare a workspace that holds n = 8 only: n = 1024 must be refused, not overrun it
        assert lib.sparc_gpu_set_workspace_size(g._ctx, g.workspace_bytes(api.OP_EIGENSOLVE, 8)) == 0
        assert lib.sparc_gpu_eigensolve(g._ctx, 1024, p, p, p, p, None, C.c_void_p(g._ws.data_ptr()), None) == -5
    finally:
        lib.sparc_gpu_set_workspace_size(g._ctx, declared)
