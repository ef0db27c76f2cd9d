"""Seeded synthetic CheFSI workloads (inputs only; no method arithmetic lives here).

This module is the ONE thing the CPU oracle (``oracle/``) and the CUDA path
(``paper_2302_09708_b200/csrc``) have in common: it manufactures the inputs both are
fed -- grid, boundary flags, atom positions, Kleinman-Bylander projector tables
(support index lists, chi, gamma), the local potential Veff, the orbital block Psi,
the rotation matrix Q and the filter bounds (a0, a, b).  None of the operators of the
hot path (stencil, H*Psi, Chebyshev recurrence, Psi^T Y, Psi Q) is implemented here.

The five named workloads follow ``BASELINE.json:configs[0..4]`` made concrete by
SURVEY.md section 8(d) ("Synthetic inputs").  They stand in for the paper's Mo / TiO2
systems (section III), whose structures and pseudopotentials are not
available; shapes follow the paper's (cubic periodic bulk grids, slab grids with
vacuum, N_s in the thousands, Chebyshev degree 10..24).

Randomness: one stateless counter-based generator ``u(seed, stream, index) in [0,1)``
(`counter_uniform`).  The CUDA library restates the same integer mix in its device
fill kernel (``sparc_gpu_fill_uniform``) so that an 82 GB Psi never crosses PCIe; the
two implementations are independent restatements of the recipe documented here.

Streams: 1 = Psi, 2 = Veff noise, 3 = atom positions / jitter, 4 = Veff centres,
5 = gamma, 6 = Q (Gaussian matrix), 7 = Veff smooth-noise parameters, 8 = imaginary part of a complex Psi,
9 = occupations.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional, Sequence, Tuple

import numpy as np

STREAM_PSI = 1
STREAM_VEFF_NOISE = 2
STREAM_ATOMS = 3
STREAM_VEFF_CENTRES = 4
STREAM_GAMMA = 5
STREAM_Q = 6
STREAM_VEFF_SMOOTH = 7
STREAM_PSI_IMAG = 8
STREAM_OCC = 9

_M64 = (1 << 64) - 1
_GOLDEN = 0x9E3779B97F4A7C15
_C_SEED = 0xD1B54A32D192ED03
_C_STREAM = 0x8CB92BA72F3D8DD7
_MIX1 = 0xBF58476D1CE4E5B9
_MIX2 = 0x94D049BB133111EB


def _mix64_int(z: int) -> int:
    z &= _M64
    z = ((z ^ (z >> 30)) * _MIX1) & _M64
    z = ((z ^ (z >> 27)) * _MIX2) & _M64
    return z ^ (z >> 31)


def stream_key(seed: int, stream: int) -> int:
    """64-bit key of a (seed, stream) pair: mix64(seed*C_SEED + stream*C_STREAM + GOLDEN)."""
    return _mix64_int((seed * _C_SEED + stream * _C_STREAM + _GOLDEN) & _M64)


def counter_uniform(seed: int, stream: int, index) -> np.ndarray:
    """u(seed, stream, index) in [0, 1): top 53 bits of mix64(key + GOLDEN*index).

    `index` may be a scalar or any integer array (treated as uint64).
    """
    key = np.uint64(stream_key(seed, stream))
    idx = np.asarray(index).astype(np.uint64)
    with np.errstate(over="ignore"):
        z = key + np.uint64(_GOLDEN) * idx
        z = (z ^ (z >> np.uint64(30))) * np.uint64(_MIX1)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(_MIX2)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def counter_uniform_range(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    return counter_uniform(seed, stream, np.arange(start, start + count, dtype=np.uint64))


# ----------------------------------------------------------------------------------
# Workload container
# ----------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    seed: int
    n: Tuple[int, int, int]            # nx, ny, nz; linear index i = x + nx*(y + ny*z)
    h: Tuple[float, float, float]      # grid spacing per axis (bohr)
    bc: Tuple[int, int, int]           # 0 = periodic, 1 = Dirichlet
    fd_order: int                      # n0 (radius = n0/2)
    ns: int                            # number of orbitals (columns of Psi)
    degree: int                        # Chebyshev degree m
    atom_pos: np.ndarray               # [n_atoms, 3] positions in bohr
    n_proj: np.ndarray                 # [n_atoms] int32, projectors per atom
    rc: float
    supp_ptr: np.ndarray               # [n_atoms+1] int64
    supp_idx: np.ndarray               # int32, ascending within each atom
    chi_ptr: np.ndarray                # [n_atoms+1] int64 offsets (doubles) into chi
    chi: np.ndarray                    # per atom n_J x P_J column-major, float64
    gamma: np.ndarray                  # concatenated P_J per atom, float64
    veff: np.ndarray                   # [Nd] float64
    a0: float = 0.0
    a: float = 0.0
    b: float = 0.0
    col_block: int = 0                 # filter column block (0 = library chooses)
    row_panel: int = 0                 # rotation row panel (0 = library chooses)
    notes: str = ""
    supp_shift: Optional[np.ndarray] = None   # [supp_total, 3] int8: cells each support row was folded by (k-point phases)

    @property
    def nd(self) -> int:
        return int(self.n[0]) * int(self.n[1]) * int(self.n[2])

    @property
    def n_atoms(self) -> int:
        return int(self.n_proj.shape[0])

    @property
    def gamma_ptr(self) -> np.ndarray:
        out = np.zeros(self.n_atoms + 1, dtype=np.int64)
        np.cumsum(self.n_proj, out=out[1:])
        return out

    @property
    def coverage(self) -> float:
        return float(self.supp_idx.shape[0]) / float(self.nd)

    # ---- Psi, Q (inputs) ----------------------------------------------------------
    def psi_columns(self, cols: Sequence[int]) -> np.ndarray:
        """Columns `cols` of Psi as an (Nd, len(cols)) Fortran-ordered array.

        Psi[i, j] = 2*u(seed, STREAM_PSI, i + Nd*j) - 1, i.i.d. U(-1, 1)."""
        nd = self.nd
        out = np.empty((nd, len(cols)), dtype=np.float64, order="F")
        base = np.arange(nd, dtype=np.uint64)
        for k, j in enumerate(cols):
            out[:, k] = 2.0 * counter_uniform(self.seed, STREAM_PSI, base + np.uint64(nd * int(j))) - 1.0
        return out

    def psi(self) -> np.ndarray:
        return self.psi_columns(range(self.ns))

    def psi_rows(self, rows: Sequence[int]) -> np.ndarray:
        """Rows `rows` (grid indices) of Psi, all ns columns, as a (len(rows), ns) Fortran-ordered array."""
        nd = self.nd
        r = np.asarray(list(rows), dtype=np.uint64)
        out = np.empty((r.shape[0], self.ns), dtype=np.float64, order="F")
        for j in range(self.ns):
            out[:, j] = 2.0 * counter_uniform(self.seed, STREAM_PSI, r + np.uint64(nd * j)) - 1.0
        return out

    def psi_columns_complex(self, cols: Sequence[int]) -> np.ndarray:
        """Complex columns for the k-point variant: real part as psi_columns, imaginary part from STREAM_PSI_IMAG."""
        nd = self.nd
        out = np.empty((nd, len(cols)), dtype=np.complex128, order="F")
        base = np.arange(nd, dtype=np.uint64)
        for k, j in enumerate(cols):
            idx = base + np.uint64(nd * int(j))
            out[:, k] = (2.0 * counter_uniform(self.seed, STREAM_PSI, idx) - 1.0) + 1j * (
                2.0 * counter_uniform(self.seed, STREAM_PSI_IMAG, idx) - 1.0)
        return out

    def occupations(self) -> np.ndarray:
        """Synthetic occupation numbers g_n in [0, 2] (spin-degenerate), decreasing with the orbital index: inputs of
        the nonlocal-force contraction."""
        u = counter_uniform_range(self.seed, STREAM_OCC, 0, self.ns)
        x = (np.arange(self.ns) + u) / max(self.ns, 1)
        return 2.0 / (1.0 + np.exp(12.0 * (x - 0.85)))

    def q_matrix(self) -> np.ndarray:
        """Haar-random orthogonal Q (ns x ns, Fortran order): Gaussian matrix -> QR -> sign fix."""
        ns = self.ns
        cnt = ns * ns
        u1 = counter_uniform_range(self.seed, STREAM_Q, 0, cnt)
        u2 = counter_uniform_range(self.seed, STREAM_Q, cnt, cnt)
        g = np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * math.pi * u2)   # Box-Muller
        g = np.asfortranarray(g.reshape(ns, ns))
        q, r = np.linalg.qr(g)
        d = np.sign(np.diag(r))
        d[d == 0] = 1.0
        return np.asfortranarray(q * d[None, :])


# ----------------------------------------------------------------------------------
# Geometry helpers (inputs: support sets and projector tables)
# ----------------------------------------------------------------------------------
def _axis_offsets(pos: float, h: float, n: int, bc: int, rc: float):
    """Grid indices (possibly wrapped) and displacements along one axis within rc of `pos`.

    Periodic axis: minimum-image displacement, indices taken mod n.
    Dirichlet axis: plain distance, indices outside [0, n-1] absent."""
    lo = int(math.floor((pos - rc) / h)) - 1
    hi = int(math.ceil((pos + rc) / h)) + 1
    k = np.arange(lo, hi + 1)
    d = k * h - pos                              # displacement grid point - atom
    if bc == 0:
        idx = np.mod(k, n)
        wrap = np.floor_divide(k, n)             # cells the true support point lies beyond the cell (image shift)
    else:
        keep = (k >= 0) & (k < n)
        k, d = k[keep], d[keep]
        idx = k
        wrap = np.zeros_like(k)
    keep = np.abs(d) <= rc + 1e-12
    return idx[keep].astype(np.int64), d[keep], wrap[keep].astype(np.int8)


def real_harmonics(dx, dy, dz, r, n_proj: int) -> np.ndarray:
    """Real spherical harmonics Y_lm(r_hat) for the first `n_proj` channels.

    Order: s | p_x, p_y, p_z | d_xy, d_yz, d_z2, d_xz, d_x2-y2 (standard normalisation).
    l > 0 channels are set to 0 at r = 0."""
    out = np.zeros((r.shape[0], n_proj), dtype=np.float64)
    out[:, 0] = 1.0 / math.sqrt(4.0 * math.pi)
    if n_proj == 1:
        return out
    safe = np.where(r > 0, r, 1.0)
    ux, uy, uz = dx / safe, dy / safe, dz / safe
    nz = r > 0
    cp = math.sqrt(3.0 / (4.0 * math.pi))
    for k, u in enumerate((ux, uy, uz)):
        if 1 + k < n_proj:
            out[:, 1 + k] = np.where(nz, cp * u, 0.0)
    if n_proj > 4:
        c15 = 0.5 * math.sqrt(15.0 / math.pi)
        c5 = 0.25 * math.sqrt(5.0 / math.pi)
        c15b = 0.25 * math.sqrt(15.0 / math.pi)
        d = [c15 * ux * uy, c15 * uy * uz, c5 * (3.0 * uz * uz - 1.0), c15 * ux * uz,
             c15b * (ux * ux - uy * uy)]
        for k, v in enumerate(d):
            if 4 + k < n_proj:
                out[:, 4 + k] = np.where(nz, v, 0.0)
    return out


def build_projectors(n, h, bc, atom_pos, n_proj, rc, width: float = 1.0):
    """Support index lists and chi tables for all atoms.

    chi_J[t, q] = exp(-r^2 / (2 width^2)) * Y_q(r_hat), r = min-image displacement of grid point
    idx_J[t] from atom J, truncated at |r| <= rc; rows ascending in grid index."""
    nx, ny, nz = n
    supp_ptr = [0]
    chi_ptr = [0]
    idx_all, chi_all, shift_all = [], [], []
    for J in range(atom_pos.shape[0]):
        P = int(n_proj[J])
        ix, dx, wx = _axis_offsets(atom_pos[J, 0], h[0], nx, bc[0], rc)
        iy, dy, wy = _axis_offsets(atom_pos[J, 1], h[1], ny, bc[1], rc)
        iz, dz, wz = _axis_offsets(atom_pos[J, 2], h[2], nz, bc[2], rc)
        DX, DY, DZ = np.meshgrid(dx, dy, dz, indexing="ij")
        IX, IY, IZ = np.meshgrid(ix, iy, iz, indexing="ij")
        WX, WY, WZ = np.meshgrid(wx, wy, wz, indexing="ij")
        r = np.sqrt(DX * DX + DY * DY + DZ * DZ).ravel()
        keep = r <= rc
        lin = (IX + nx * (IY + ny * IZ)).ravel()[keep]
        dxk, dyk, dzk, rk = DX.ravel()[keep], DY.ravel()[keep], DZ.ravel()[keep], r[keep]
        order = np.argsort(lin, kind="stable")
        lin, dxk, dyk, dzk, rk = lin[order], dxk[order], dyk[order], dzk[order], rk[order]
        shift_all.append(np.stack([WX.ravel()[keep][order], WY.ravel()[keep][order], WZ.ravel()[keep][order]], axis=1))
        if lin.size > 1 and np.any(np.diff(lin) == 0):
            raise ValueError("atom support wraps onto itself (need 2*rc < L on periodic axes)")
        radial = np.exp(-(rk * rk) / (2.0 * width * width))
        table = radial[:, None] * real_harmonics(dxk, dyk, dzk, rk, P)    # n_J x P
        idx_all.append(lin.astype(np.int32))
        chi_all.append(np.asfortranarray(table).ravel(order="F"))
        supp_ptr.append(supp_ptr[-1] + lin.size)
        chi_ptr.append(chi_ptr[-1] + lin.size * P)
    supp_idx = np.concatenate(idx_all) if idx_all else np.zeros(0, np.int32)
    chi = np.concatenate(chi_all) if chi_all else np.zeros(0, np.float64)
    shift = np.concatenate(shift_all).astype(np.int8) if shift_all else np.zeros((0, 3), np.int8)
    return (np.asarray(supp_ptr, np.int64), supp_idx.astype(np.int32),
            np.asarray(chi_ptr, np.int64), chi.astype(np.float64), shift)


def _min_image(d, L, periodic: bool):
    if periodic:
        return d - L * np.round(d / L)
    return d


def gaussian_wells(n, h, bc, centres, depth=-2.0, width=1.5) -> np.ndarray:
    """sum_R depth*exp(-|r-R|^2/(2 width^2)) on the grid (min-image on periodic axes)."""
    nx, ny, nz = n
    L = (nx * h[0], ny * h[1], nz * h[2])
    x = np.arange(nx) * h[0]
    y = np.arange(ny) * h[1]
    z = np.arange(nz) * h[2]
    v = np.zeros((nz, ny, nx), dtype=np.float64)
    inv = 1.0 / (2.0 * width * width)
    for R in centres:
        ex = np.exp(-_min_image(x - R[0], L[0], bc[0] == 0) ** 2 * inv)
        ey = np.exp(-_min_image(y - R[1], L[1], bc[1] == 0) ** 2 * inv)
        ez = np.exp(-_min_image(z - R[2], L[2], bc[2] == 0) ** 2 * inv)
        v += depth * ez[:, None, None] * ey[None, :, None] * ex[None, None, :]
    return v.ravel()


# |w_0| + 2 sum_p |w_p| of the radius-6 central second-derivative weights = 367616/51975
# (SURVEY.md section 8(c) R18).  Used ONLY to manufacture the input bound b.
_STENCIL_ABS_SUM_R6 = 367616.0 / 51975.0


def _stencil_abs_sum(fd_order: int) -> float:
    if fd_order == 12:
        return _STENCIL_ABS_SUM_R6
    # generic: |w0| + 2 sum |w_p| from the closed form of the central weights
    r = fd_order // 2
    s = 0.0
    w0 = 0.0
    for p in range(1, r + 1):
        wp = 2.0 * (-1.0) ** (p + 1) / (p * p) * (math.factorial(r) ** 2) / (
            math.factorial(r - p) * math.factorial(r + p))
        s += 2.0 * abs(wp)
        w0 -= 2.0 / (p * p)
    return s + abs(w0)


def filter_bounds(n, h, fd_order, veff, supp_ptr, supp_idx, chi_ptr, chi, gamma, n_proj):
    """(a0, a, b) per BASELINE.json:configs[0] / SURVEY R18.

    b  = 1/2 sum_axis S/h_axis^2 + max(Veff) + B_nl, S = stencil abs-sum;
    B_nl = K * max_J sum_q max(gamma_Jq, 0) * ||chi_Jq||_2^2, K = max number of supports per point;
    a0 = min(Veff);  a = a0 + 0.3 (b - a0).  These are INPUTS handed to both sides."""
    S = _stencil_abs_sum(fd_order)
    kin = 0.5 * sum(S / (hh * hh) for hh in h)
    nd = int(n[0]) * int(n[1]) * int(n[2])
    cover = np.bincount(supp_idx.astype(np.int64), minlength=nd) if supp_idx.size else np.zeros(1)
    K = float(cover.max()) if supp_idx.size else 0.0
    bmax = 0.0
    g0 = 0
    for J in range(len(n_proj)):
        P = int(n_proj[J])
        nJ = int(supp_ptr[J + 1] - supp_ptr[J])
        tab = chi[chi_ptr[J]:chi_ptr[J + 1]].reshape((nJ, P), order="F")
        gam = gamma[g0:g0 + P]
        g0 += P
        val = float(np.sum(np.maximum(gam, 0.0) * np.sum(tab * tab, axis=0)))
        bmax = max(bmax, val)
    b = kin + float(veff.max()) + K * bmax
    a0 = float(veff.min())
    a = a0 + 0.3 * (b - a0)
    return a0, a, b


# ----------------------------------------------------------------------------------
# Named workloads
# ----------------------------------------------------------------------------------
def _uniform_positions(seed, count, L):
    u = counter_uniform_range(seed, STREAM_ATOMS, 0, 3 * count).reshape(count, 3)
    return u * np.asarray(L)[None, :]


def _lattice_positions(seed, cells, basis, origin, span, jitter):
    """Sites of a (cells[0] x cells[1] x cells[2]) lattice with fractional `basis`, filling the box
    origin .. origin+span, jittered by U(-jitter, jitter) per coordinate."""
    sites = []
    for k in range(cells[2]):
        for j in range(cells[1]):
            for i in range(cells[0]):
                for bvec in basis:
                    sites.append(((i + bvec[0]) / cells[0], (j + bvec[1]) / cells[1],
                                  (k + bvec[2]) / cells[2]))
    sites = np.asarray(sites, dtype=np.float64)
    pos = np.asarray(origin)[None, :] + sites * np.asarray(span)[None, :]
    u = counter_uniform_range(seed, STREAM_ATOMS, 0, pos.size).reshape(pos.shape)
    return pos + jitter * (2.0 * u - 1.0)


def _smooth_noise(seed, n, h):
    """8 cosines with integer wavevectors |n_i| <= 2, amplitudes U(-0.05,0.05), random phases."""
    nx, ny, nz = n
    u = counter_uniform_range(seed, STREAM_VEFF_SMOOTH, 0, 8 * 5).reshape(8, 5)
    x = np.arange(nx) / nx
    y = np.arange(ny) / ny
    z = np.arange(nz) / nz
    v = np.zeros((nz, ny, nx))
    for t in range(8):
        kx, ky, kz = (np.floor(u[t, :3] * 5.0) - 2.0).astype(int)
        amp = 0.05 * (2.0 * u[t, 3] - 1.0)
        ph = 2.0 * math.pi * u[t, 4]
        arg = 2.0 * math.pi * (kx * x[None, None, :] + ky * y[None, :, None] + kz * z[:, None, None]) + ph
        v += amp * np.cos(arg)
    return v.ravel()


_SC = ((0.5, 0.5, 0.5),)
_FCC = ((0.25, 0.25, 0.25), (0.75, 0.75, 0.25), (0.75, 0.25, 0.75), (0.25, 0.75, 0.75))

CONFIG_TABLE = {
    0: dict(name="cfg0_tiny_periodic_24", n=(24, 24, 24), h=0.5, bc=(0, 0, 0), ns=32, degree=10,
            atoms=4, P=4, rc=3.0),
    1: dict(name="cfg1_bulk_periodic_48", n=(48, 48, 48), h=0.4, bc=(0, 0, 0), ns=256, degree=20,
            atoms=32, P=4, rc=3.0),
    2: dict(name="cfg2_slab_60x60x180", n=(60, 60, 180), h=0.35, bc=(0, 0, 1), ns=1024, degree=16,
            atoms=128, P=9, rc=3.5),
    3: dict(name="cfg3_bulk_96", n=(96, 96, 96), h=0.3, bc=(0, 0, 0), ns=4096, degree=20,
            atoms=512, P=9, rc=3.5),
    4: dict(name="cfg4_metallic_96x96x144", n=(96, 96, 144), h=0.3, bc=(0, 0, 0), ns=7680, degree=24,
            atoms=1000, P=9, rc=3.5, col_block=1024),
    # sixth workload: the paper's finer-mesh regime, h = 0.22 bohr and Chebyshev degree 33
    # (PAPER.md:182), on a grid one GPU holds
    5: dict(name="cfg5_fine_mesh_128", n=(128, 128, 128), h=0.22, bc=(0, 0, 0), ns=2048, degree=33,
            atoms=216, P=9, rc=3.5, col_block=1024),
}


def make_workload(config: int, ns: Optional[int] = None) -> Workload:
    """Workload `config` in 0..4 (BASELINE.json:configs) or 5 (the finer-mesh, degree-33 regime); seed = config number.

    `ns` overrides the orbital count (used by bounded CPU samples; Psi columns are
    position-independent streams, so a prefix of columns is the same data)."""
    c = CONFIG_TABLE[config]
    seed = config
    n = c["n"]
    h = (c["h"],) * 3
    bc = c["bc"]
    L = tuple(n[i] * h[i] for i in range(3))
    if config == 0:
        pos = _uniform_positions(seed, c["atoms"], L)
        u = counter_uniform_range(seed, STREAM_VEFF_CENTRES, 0, 12).reshape(4, 3)
        centres = u * np.asarray(L)[None, :]
    elif config == 1:
        pos = _lattice_positions(seed, (4, 4, 2), _SC, (0, 0, 0), L, 0.3)
        centres = pos
    elif config == 2:
        pos = _lattice_positions(seed, (4, 4, 8), _SC, (0, 0, 0.3 * L[2]), (L[0], L[1], 0.4 * L[2]), 0.3)
        centres = pos
    elif config == 3:
        pos = _lattice_positions(seed, (8, 8, 8), _SC, (0, 0, 0), L, 0.3)
        centres = pos
    elif config == 4:
        pos = _lattice_positions(seed, (5, 5, 10), _FCC, (0, 0, 0), L, 0.3)
        centres = pos
    elif config == 5:
        pos = _lattice_positions(seed, (6, 6, 6), _SC, (0, 0, 0), L, 0.3)
        centres = pos
    else:
        raise KeyError(config)
    # wrap periodic coordinates into the cell (positions are inputs; wrapping is cosmetic)
    for ax in range(3):
        if bc[ax] == 0:
            pos[:, ax] = np.mod(pos[:, ax], L[ax])
    n_proj = np.full(c["atoms"], c["P"], dtype=np.int32)
    supp_ptr, supp_idx, chi_ptr, chi, supp_shift = build_projectors(n, h, bc, pos, n_proj, c["rc"], 1.0)
    gamma = 2.0 * counter_uniform_range(seed, STREAM_GAMMA, 0, int(n_proj.sum())) - 1.0
    veff = gaussian_wells(n, h, bc, centres, -2.0, 1.5)
    nd = n[0] * n[1] * n[2]
    if config == 0:
        veff = veff + 0.05 * (2.0 * counter_uniform_range(seed, STREAM_VEFF_NOISE, 0, nd) - 1.0)
    elif config in (1, 3, 4, 5):
        veff = veff + _smooth_noise(seed, n, h)
    elif config == 2:
        z = (np.arange(n[2]) * h[2])[:, None, None] + np.zeros((1, n[1], n[0]))
        veff = veff + 0.01 * (z.ravel() - 0.5 * L[2])
    a0, a, b = filter_bounds(n, h, 12, veff, supp_ptr, supp_idx, chi_ptr, chi, gamma, n_proj)
    return Workload(name=c["name"], seed=seed, n=n, h=h, bc=bc, fd_order=12,
                    ns=int(ns if ns is not None else c["ns"]), degree=c["degree"], atom_pos=pos,
                    n_proj=n_proj, rc=c["rc"], supp_ptr=supp_ptr, supp_idx=supp_idx, chi_ptr=chi_ptr,
                    chi=chi, gamma=gamma, veff=np.ascontiguousarray(veff), a0=a0, a=a, b=b,
                    col_block=c.get("col_block", 0), supp_shift=supp_shift)


def make_custom(name, n, h, bc, ns, degree, atom_pos, n_proj, rc, seed=1234, fd_order=12,
                veff_kind="wells+noise", gamma=None) -> Workload:
    """Free-form small workload for tests (tiny anisotropic / mixed-BC grids, single atoms ...)."""
    n = tuple(int(v) for v in n)
    h = tuple(float(v) for v in h)
    bc = tuple(int(v) for v in bc)
    atom_pos = np.asarray(atom_pos, dtype=np.float64).reshape(-1, 3)
    n_proj = np.asarray(n_proj, dtype=np.int32).reshape(-1)
    supp_ptr, supp_idx, chi_ptr, chi, supp_shift = build_projectors(n, h, bc, atom_pos, n_proj, rc, 1.0)
    if gamma is None:
        gamma = 2.0 * counter_uniform_range(seed, STREAM_GAMMA, 0, int(n_proj.sum())) - 1.0
    gamma = np.asarray(gamma, dtype=np.float64)
    nd = n[0] * n[1] * n[2]
    if veff_kind == "zero":
        veff = np.zeros(nd)
    elif veff_kind.startswith("const:"):
        veff = np.full(nd, float(veff_kind.split(":")[1]))
    else:
        centres = atom_pos if atom_pos.shape[0] else np.zeros((0, 3))
        veff = gaussian_wells(n, h, bc, centres, -2.0, 1.5)
        veff = veff + 0.05 * (2.0 * counter_uniform_range(seed, STREAM_VEFF_NOISE, 0, nd) - 1.0)
    a0, a, b = filter_bounds(n, h, fd_order, veff, supp_ptr, supp_idx, chi_ptr, chi, gamma, n_proj)
    if not (a0 < a < b):
        a0, a = a0 - 1.0, a0 - 1.0 + 0.3 * (b - a0 + 1.0)
    return Workload(name=name, seed=seed, n=n, h=h, bc=bc, fd_order=fd_order, ns=ns, degree=degree,
                    atom_pos=atom_pos, n_proj=n_proj, rc=rc, supp_ptr=supp_ptr, supp_idx=supp_idx,
                    chi_ptr=chi_ptr, chi=chi, gamma=gamma, veff=np.ascontiguousarray(veff),
                    a0=a0, a=a, b=b, supp_shift=supp_shift)
