"""Thin Python binding of the sparc_gpu C-ABI library (include/sparc_gpu.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; PyTorch is used here for device
memory (tensors, workspaces) and streams only.  There is no CPU fallback: if libsparc_gpu.so cannot be
loaded (and cannot be built), importing/using this module raises.

Matrix convention: an N_d x ncols column-major matrix with leading dimension ld is held as a torch
float64 CUDA tensor of shape (ncols, ld) that is contiguous along its last axis (so `t[j, :N_d]` is
column j).  Helpers `colmajor_from_numpy` / `colmajor_to_numpy` convert from / to Fortran-ordered numpy.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libsparc_gpu.so")
_lib = None

OP_HAMILTONIAN_APPLY, OP_CHEBYSHEV_FILTER, OP_PROJECT, OP_ROTATE = 0, 1, 2, 3
OP_GRADIENT_PROJECT, OP_NONLOCAL_FORCE, OP_EIGENSOLVE = 4, 5, 6
OP_HAMILTONIAN_APPLY_K, OP_CHEBYSHEV_FILTER_K, OP_PROJECT_K, OP_ROTATE_K = 7, 8, 9, 10
OP_GRAM = 11

EXPORTS = ["sparc_gpu_create", "sparc_gpu_destroy", "sparc_gpu_set_veff", "sparc_gpu_workspace_bytes",
           "sparc_gpu_set_workspace_size",
           "sparc_gpu_hamiltonian_apply", "sparc_gpu_chebyshev_filter", "sparc_gpu_project",
           "sparc_gpu_rotate", "sparc_gpu_chefsi_step_host", "sparc_gpu_chefsi_step_host_solve", "sparc_gpu_gradient",
           "sparc_gpu_nl_project", "sparc_gpu_gradient_project", "sparc_gpu_nonlocal_force", "sparc_gpu_eigensolve", "sparc_gpu_set_kpoint",
           "sparc_gpu_hamiltonian_apply_k", "sparc_gpu_chebyshev_filter_k", "sparc_gpu_project_k", "sparc_gpu_rotate_k",
           "sparc_gpu_gram", "sparc_gpu_rotate_rows", "sparc_gpu_gram_static", "sparc_gpu_fill_uniform", "sparc_gpu_set_option", "sparc_gpu_get_info", "sparc_gpu_probe_peak",
           "sparc_gpu_error_string", "sparc_gpu_version"]


class SparcGpuError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = load_library().sparc_gpu_error_string(code).decode()
        super().__init__(f"{where}: {msg} (status {code})")


class Desc(C.Structure):
    _fields_ = [("n", C.c_int32 * 3), ("h", C.c_double * 3), ("bc", C.c_int32 * 3),
                ("fd_order", C.c_int32), ("n_atoms", C.c_int32),
                ("supp_ptr", C.c_void_p), ("supp_idx", C.c_void_p), ("n_proj", C.c_void_p),
                ("chi_ptr", C.c_void_p), ("chi", C.c_void_p), ("gamma", C.c_void_p),
                ("veff", C.c_void_p), ("device", C.c_int32)]


def load_library(build_if_missing: bool = True):
    """dlopen libsparc_gpu.so (building it in-tree with nvcc if absent).  Raises if impossible."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        if not build_if_missing:
            raise RuntimeError(f"{_LIB_PATH} is missing: run `python -m paper_2302_09708_b200.build`")
        from . import build as _build
        _build.build()
    lib = C.CDLL(_LIB_PATH)
    P, I64, D, I = C.c_void_p, C.c_int64, C.c_double, C.c_int
    lib.sparc_gpu_create.argtypes = [C.POINTER(Desc), C.POINTER(P)]
    lib.sparc_gpu_destroy.argtypes = [P]
    lib.sparc_gpu_set_veff.argtypes = [P, P, P]
    lib.sparc_gpu_workspace_bytes.argtypes = [P, I, I64, I64, C.POINTER(I64)]
    lib.sparc_gpu_set_workspace_size.argtypes = [P, I64]
    lib.sparc_gpu_hamiltonian_apply.argtypes = [P, P, I64, P, I64, I64, P, P]
    lib.sparc_gpu_chebyshev_filter.argtypes = [P, P, I64, I64, I, D, D, D, I64, P, P]
    lib.sparc_gpu_project.argtypes = [P, P, I64, I64, P, P, I64, P, P]
    lib.sparc_gpu_rotate.argtypes = [P, P, I64, I64, P, I64, P, P]
    lib.sparc_gpu_chefsi_step_host.argtypes = [P, P, P, I64, I64, I, D, D, D, P, P, P, P, I64, P, I64, I64, P, P]
    lib.sparc_gpu_chefsi_step_host_solve.argtypes = [P, P, P, I64, I64, I, D, D, D, P, P, P, P, P, I64, P, I64, I64, P, P]
    lib.sparc_gpu_gradient.argtypes = [P, I, P, I64, P, I64, I64, P]
    lib.sparc_gpu_nl_project.argtypes = [P, P, I64, I64, P, P]
    lib.sparc_gpu_gradient_project.argtypes = [P, I, P, I64, I64, P, I64, P, P]
    lib.sparc_gpu_nonlocal_force.argtypes = [P, P, I64, I64, P, P, I64, P, P]
    lib.sparc_gpu_eigensolve.argtypes = [P, I64, P, P, P, P, P, P, P]
    lib.sparc_gpu_set_kpoint.argtypes = [P, P, P]
    lib.sparc_gpu_hamiltonian_apply_k.argtypes = [P, P, I64, P, I64, I64, P, P]
    lib.sparc_gpu_chebyshev_filter_k.argtypes = [P, P, I64, I64, I, D, D, D, I64, P, P]
    lib.sparc_gpu_project_k.argtypes = [P, P, I64, I64, P, P, I64, P, P]
    lib.sparc_gpu_rotate_k.argtypes = [P, P, I64, I64, P, I64, P, P]
    lib.sparc_gpu_gram.argtypes = [P, P, I64, P, I64, I64, I64, I64, P, I, P, P]
    lib.sparc_gpu_rotate_rows.argtypes = [P, P, I64, I64, I64, P, I64, P, P]
    lib.sparc_gpu_gram_static.argtypes = [I, P, I64, P, I64, I64, I64, I64, P, I, P]
    lib.sparc_gpu_fill_uniform.argtypes = [P, I64, C.c_uint64, C.c_uint64, C.c_uint64, D, D, I, P]
    lib.sparc_gpu_probe_peak.argtypes = [I, I, C.POINTER(D), P, I64, P]
    lib.sparc_gpu_set_option.argtypes = [P, C.c_char_p, I64]
    lib.sparc_gpu_get_info.argtypes = [P, C.c_char_p, C.POINTER(I64)]
    lib.sparc_gpu_error_string.argtypes = [I]
    lib.sparc_gpu_error_string.restype = C.c_char_p
    lib.sparc_gpu_version.restype = C.c_char_p
    for name in EXPORTS[:-2]:
        getattr(lib, name).restype = I
    _lib = lib
    return lib


def _check(code: int, where: str):
    if code != 0:
        raise SparcGpuError(code, where)


def _torch():
    import torch
    return torch


def _stream_ptr(device=None):
    """cudaStream_t of torch's current stream ON `device` (not on whatever device happens to be current)."""
    return C.c_void_p(_torch().cuda.current_stream(device).cuda_stream)


def colmajor_from_numpy(a: np.ndarray, device="cuda", ld: Optional[int] = None):
    """(rows x cols) numpy array -> torch (cols, ld) float64 CUDA tensor holding it column-major."""
    torch = _torch()
    a = np.asarray(a, dtype=np.float64)
    if a.ndim == 1:
        a = a.reshape(-1, 1)
    rows, cols = a.shape
    ld = rows if ld is None else int(ld)
    t = torch.zeros((cols, ld), dtype=torch.float64, device=device)
    t[:, :rows] = torch.from_numpy(np.ascontiguousarray(a.T)).to(device)
    return t


def colmajor_to_numpy(t, rows: Optional[int] = None) -> np.ndarray:
    rows = t.shape[1] if rows is None else rows
    return np.asfortranarray(t[:, :rows].detach().cpu().numpy().T)


def fill_uniform(t, seed: int, stream_id: int, index0: int, lo: float, hi: float):
    """t.view(-1)[k] = lo + (hi-lo)*u(seed, stream_id, index0+k) on the device (contiguous tensor)."""
    assert t.is_cuda and t.is_contiguous() and t.dtype == _torch().float64
    _check(load_library().sparc_gpu_fill_uniform(C.c_void_p(t.data_ptr()), t.numel(), seed, stream_id, index0,
                                                 lo, hi, t.device.index or 0, _stream_ptr(t.device)), "fill_uniform")
    return t


def probe_peak(kind: int, device: int = 0, scratch_bytes: int = 1 << 30) -> float:
    """kind 0: FP64 FMA TFLOP/s, 1: FP64 DMMA TFLOP/s, 2: device copy GB/s -- measured live (sparc_gpu_probe_peak)."""
    torch = _torch()
    scratch = torch.empty(scratch_bytes if kind == 2 else 4096, dtype=torch.uint8, device=f"cuda:{device}")
    out = C.c_double()
    _check(load_library().sparc_gpu_probe_peak(int(device), int(kind), C.byref(out), C.c_void_p(scratch.data_ptr()),
                                               scratch.numel(), _stream_ptr(scratch.device)), "probe_peak")
    return out.value


GRAM_STATIC_MAX_ELEMS = 2097152       # SPARC_GPU_GRAM_STATIC_MAX_ELEMS of include/sparc_gpu.h


def gram_static(A, B, nrows: int, symmetric: bool = False, out=None):
    """sparc_gpu_gram_static: C = A^T B over `nrows` rows without a context, a workspace or any device allocation by the
    library -- for callers that cannot allocate at this point (all HBM already in their own arena or under a per-process
    cap; inside an overlapped multi-stream region that a cudaMalloc / cudaFree would stall; memory owned by a host
    application's allocator).  The split-K partials live in a 16 MiB array built into the library, one per GPU and shared by
    all calls: keep calls on one stream or order them with events.  m * n <= GRAM_STATIC_MAX_ELEMS, else SparcGpuError
    (status -8).  A, B: (m, lda), (n, ldb) float64 CUDA tensors holding the column-major nrows x m / nrows x n matrices.
    Pass `out` ((n, m), contiguous) if this wrapper must not allocate either; the first call on a device does a one-time
    address look-up and belongs before any stream capture.  Runs on torch's current stream of A's device."""
    torch = _torch()
    for t in (A, B):
        if not (t.is_cuda and t.dtype == torch.float64 and t.dim() == 2 and t.stride(1) == 1):
            raise ValueError("gram_static: need 2-D float64 CUDA tensors (ncols, ld) contiguous along ld")
    m, n = int(A.shape[0]), int(B.shape[0])
    lda = int(A.stride(0)) if m > 1 else int(A.shape[1])
    ldb = int(B.stride(0)) if n > 1 else int(B.shape[1])
    if out is None:
        out = torch.empty((n, m), dtype=torch.float64, device=A.device)
    assert out.is_cuda and out.dtype == torch.float64 and out.shape == (n, m) and out.is_contiguous()
    dev = A.device.index if A.device.index is not None else torch.cuda.current_device()
    _check(load_library().sparc_gpu_gram_static(int(dev), C.c_void_p(A.data_ptr()), lda, C.c_void_p(B.data_ptr()), ldb,
                                                int(nrows), m, n, C.c_void_p(out.data_ptr()), 1 if symmetric else 0,
                                                _stream_ptr(A.device)), "gram_static")
    return out          # (n, m) tensor holding the column-major m x n matrix


class SparcGpu:
    """One sparc_gpu context: H = -1/2 Laplacian + Veff + V_nl on a fixed grid (see include/sparc_gpu.h)."""

    def __init__(self, wl, device: int = 0, upload_veff: bool = True):
        """`wl`: object with attributes n, h, bc, fd_order, supp_ptr, supp_idx, n_proj, chi_ptr, chi, gamma,
        veff (numpy arrays; e.g. workloads.Workload)."""
        torch = _torch()
        if not torch.cuda.is_available():
            raise RuntimeError("sparc_gpu needs a CUDA device (no CPU fallback)")
        self.lib = load_library()
        self.device = int(device)
        self.nd = int(wl.n[0]) * int(wl.n[1]) * int(wl.n[2])
        keep = dict(
            supp_ptr=np.ascontiguousarray(wl.supp_ptr, dtype=np.int64),
            supp_idx=np.ascontiguousarray(wl.supp_idx, dtype=np.int32),
            n_proj=np.ascontiguousarray(wl.n_proj, dtype=np.int32),
            chi_ptr=np.ascontiguousarray(wl.chi_ptr, dtype=np.int64),
            chi=np.ascontiguousarray(wl.chi, dtype=np.float64),
            gamma=np.ascontiguousarray(wl.gamma, dtype=np.float64))
        d = Desc()
        for k in range(3):
            d.n[k], d.h[k], d.bc[k] = int(wl.n[k]), float(wl.h[k]), int(wl.bc[k])
        d.fd_order = int(wl.fd_order)
        d.n_atoms = int(keep["n_proj"].shape[0])
        self.n_atoms = d.n_atoms
        for name, arr in keep.items():
            setattr(d, name, arr.ctypes.data if arr.size else None)
        veff = None
        if upload_veff and getattr(wl, "veff", None) is not None:
            veff = np.ascontiguousarray(wl.veff, dtype=np.float64)
            assert veff.shape[0] == self.nd
            d.veff = veff.ctypes.data
        d.device = self.device
        self._ctx = C.c_void_p()
        torch.cuda.init()
        _check(self.lib.sparc_gpu_create(C.byref(d), C.byref(self._ctx)), "sparc_gpu_create")
        self._ws = None

    # ---- lifetime -----------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self.lib.sparc_gpu_destroy(self._ctx)
            self._ctx = C.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- plumbing -----------------------------------------------------------------------------
    def workspace_bytes(self, op: int, ns: int, block: int = 0) -> int:
        out = C.c_int64()
        _check(self.lib.sparc_gpu_workspace_bytes(self._ctx, op, ns, block, C.byref(out)), "workspace_bytes")
        return out.value

    def _workspace(self, op: int, ns: int, block: int):
        torch = _torch()
        need = self.workspace_bytes(op, ns, block)
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self._ws = torch.empty(need, dtype=torch.uint8, device=f"cuda:{self.device}")
            # the ABI carries no size with ws_dev: declare it, so that a short buffer is an error code, not an overrun
            _check(self.lib.sparc_gpu_set_workspace_size(self._ctx, self._ws.numel()), "set_workspace_size")
        return C.c_void_p(self._ws.data_ptr())

    def release_workspace(self):
        self._ws = None
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self.lib.sparc_gpu_set_workspace_size(self._ctx, 0)

    def _stream(self):
        return _stream_ptr(self.device)

    def set_option(self, key: str, value: int):
        _check(self.lib.sparc_gpu_set_option(self._ctx, key.encode(), int(value)), f"set_option({key})")

    def get_info(self, key: str) -> int:
        out = C.c_int64()
        _check(self.lib.sparc_gpu_get_info(self._ctx, key.encode(), C.byref(out)), f"get_info({key})")
        return out.value

    def _mat(self, t, name: str) -> Tuple[C.c_void_p, int, int]:
        torch = _torch()
        if not (t.is_cuda and t.dtype == torch.float64 and t.dim() == 2 and t.stride(1) == 1):
            raise ValueError(f"{name}: need a 2-D float64 CUDA tensor (ncols, ld) contiguous along ld")
        if t.shape[1] < self.nd:
            raise ValueError(f"{name}: ld {t.shape[1]} < N_d {self.nd}")
        return C.c_void_p(t.data_ptr()), int(t.stride(0)) if t.shape[0] > 1 else int(t.shape[1]), int(t.shape[0])

    # ---- the C-ABI calls ----------------------------------------------------------------------
    def set_veff(self, veff):
        assert veff.is_cuda and veff.numel() >= self.nd and veff.is_contiguous()
        _check(self.lib.sparc_gpu_set_veff(self._ctx, C.c_void_p(veff.data_ptr()), self._stream()), "set_veff")

    def hamiltonian_apply(self, X, Y=None):
        torch = _torch()
        xp, ldx, ncols = self._mat(X, "X")
        if Y is None:
            Y = torch.empty_like(X)
        yp, ldy, _ = self._mat(Y, "Y")
        ws = self._workspace(OP_HAMILTONIAN_APPLY, ncols, 0)
        _check(self.lib.sparc_gpu_hamiltonian_apply(self._ctx, xp, ldx, yp, ldy, ncols, ws, self._stream()),
               "hamiltonian_apply")
        return Y

    def chebyshev_filter(self, Psi, degree: int, a: float, b: float, a0: float, col_block: int = 0):
        pp, ld, ns = self._mat(Psi, "Psi")
        ws = self._workspace(OP_CHEBYSHEV_FILTER, ns, col_block)
        _check(self.lib.sparc_gpu_chebyshev_filter(self._ctx, pp, ld, ns, int(degree), float(a), float(b),
                                                   float(a0), int(col_block), ws, self._stream()),
               "chebyshev_filter")
        return Psi

    def chefsi_step_host(self, host_psi, Q_host, Hs_host, Ms_host, degree: int, a: float, b: float, a0: float,
                         psi_dev=None, mats_dev=None, col_block: int = 0, row_panel: int = 0, host_out=None):
        """sparc_gpu_chefsi_step_host: filter -> project -> rotate on a block in (pinned) HOST memory.  host_psi:
        (ns, ld) CPU tensor, overwritten with the rotated block unless host_out is given; Q_host, Hs_host, Ms_host: (ns, ns)
        CPU tensors.  psi_dev / mats_dev: optional device scratch to reuse.  Synchronises."""
        torch = _torch()
        ns, ld = int(host_psi.shape[0]), int(host_psi.shape[1])
        host_out = host_psi if host_out is None else host_out
        for t in (host_psi, host_out, Q_host, Hs_host, Ms_host):
            assert (not t.is_cuda) and t.dtype == torch.float64 and t.is_contiguous()
        assert ld >= self.nd and host_out.shape == host_psi.shape and Q_host.shape == (ns, ns)
        dev = torch.device("cuda", self.device)
        if psi_dev is None:
            psi_dev = torch.empty((ns, self.nd), dtype=torch.float64, device=dev)
        if mats_dev is None:
            mats_dev = torch.empty(3 * ns * ns, dtype=torch.float64, device=dev)
        pp, ldd, _ = self._mat(psi_dev, "psi_dev")
        need = max(self.workspace_bytes(OP_CHEBYSHEV_FILTER, ns, col_block), self.workspace_bytes(OP_PROJECT, ns, col_block),
                   self.workspace_bytes(OP_ROTATE, ns, row_panel))
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self._ws = torch.empty(need, dtype=torch.uint8, device=dev)
            _check(self.lib.sparc_gpu_set_workspace_size(self._ctx, self._ws.numel()), "set_workspace_size")
        _check(self.lib.sparc_gpu_chefsi_step_host(
            self._ctx, C.c_void_p(host_psi.data_ptr()), C.c_void_p(host_out.data_ptr()), ld, ns, int(degree), float(a),
            float(b), float(a0), C.c_void_p(Q_host.data_ptr()), C.c_void_p(Hs_host.data_ptr()),
            C.c_void_p(Ms_host.data_ptr()), pp, ldd, C.c_void_p(mats_dev.data_ptr()), int(col_block), int(row_panel),
            C.c_void_p(self._ws.data_ptr()), self._stream()), "chefsi_step_host")
        return host_out

    def chefsi_step_host_solve(self, host_psi, Hs_host, Ms_host, degree: int, a: float, b: float, a0: float,
                               psi_dev=None, mats_dev=None, col_block: int = 0, row_panel: int = 0, host_out=None):
        """sparc_gpu_chefsi_step_host_solve: filter -> project -> device eigensolve -> rotate on a block in (pinned) HOST
        memory (Algorithm 1 with no caller-supplied Q).  Returns (host_out, D (ns,) CPU tensor, info (2,) int32 CPU tensor)."""
        torch = _torch()
        ns, ld = int(host_psi.shape[0]), int(host_psi.shape[1])
        host_out = host_psi if host_out is None else host_out
        for t in (host_psi, host_out, Hs_host, Ms_host):
            assert (not t.is_cuda) and t.dtype == torch.float64 and t.is_contiguous()
        assert ld >= self.nd and host_out.shape == host_psi.shape
        dev = torch.device("cuda", self.device)
        if psi_dev is None:
            psi_dev = torch.empty((ns, self.nd), dtype=torch.float64, device=dev)
        if mats_dev is None:
            mats_dev = torch.empty(3 * ns * ns + ns + 1, dtype=torch.float64, device=dev)
        assert mats_dev.numel() >= 3 * ns * ns + ns + 1
        pp, ldd, _ = self._mat(psi_dev, "psi_dev")
        need = max(self.workspace_bytes(OP_CHEBYSHEV_FILTER, ns, col_block), self.workspace_bytes(OP_PROJECT, ns, col_block),
                   self.workspace_bytes(OP_ROTATE, ns, row_panel), self.workspace_bytes(OP_EIGENSOLVE, ns, 0))
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self._ws = torch.empty(need, dtype=torch.uint8, device=dev)
            _check(self.lib.sparc_gpu_set_workspace_size(self._ctx, self._ws.numel()), "set_workspace_size")
        D = torch.empty(ns, dtype=torch.float64).pin_memory()
        info = torch.zeros(2, dtype=torch.int32).pin_memory()
        _check(self.lib.sparc_gpu_chefsi_step_host_solve(
            self._ctx, C.c_void_p(host_psi.data_ptr()), C.c_void_p(host_out.data_ptr()), ld, ns, int(degree), float(a),
            float(b), float(a0), C.c_void_p(D.data_ptr()), C.c_void_p(info.data_ptr()), C.c_void_p(Hs_host.data_ptr()),
            C.c_void_p(Ms_host.data_ptr()), pp, ldd, C.c_void_p(mats_dev.data_ptr()), int(col_block), int(row_panel),
            C.c_void_p(self._ws.data_ptr()), self._stream()), "chefsi_step_host_solve")
        return host_out, D, info

    # ---- NEXT-3: gradient stencil, projector contraction, nonlocal force --------------------------
    def gradient(self, X, axis: int, Y=None):
        torch = _torch()
        xp, ldx, ncols = self._mat(X, "X")
        if Y is None:
            Y = torch.empty_like(X)
        yp, ldy, _ = self._mat(Y, "Y")
        _check(self.lib.sparc_gpu_gradient(self._ctx, int(axis), xp, ldx, yp, ldy, ncols, self._stream()), "gradient")
        return Y

    def nl_project(self, X):
        """W = chi^T X as an (ncols, n_proj_total) tensor holding the column-major n_proj_total x ncols matrix."""
        torch = _torch()
        xp, ldx, ncols = self._mat(X, "X")
        W = torch.zeros((ncols, self.get_info("n_proj_total")), dtype=torch.float64, device=X.device)
        _check(self.lib.sparc_gpu_nl_project(self._ctx, xp, ldx, ncols, C.c_void_p(W.data_ptr()), self._stream()), "nl_project")
        return W

    def gradient_project(self, X, axis: int, col_block: int = 0):
        torch = _torch()
        xp, ldx, ncols = self._mat(X, "X")
        W = torch.zeros((ncols, self.get_info("n_proj_total")), dtype=torch.float64, device=X.device)
        ws = self._workspace(OP_GRADIENT_PROJECT, ncols, col_block)
        _check(self.lib.sparc_gpu_gradient_project(self._ctx, int(axis), xp, ldx, ncols, C.c_void_p(W.data_ptr()),
                                                   int(col_block), ws, self._stream()), "gradient_project")
        return W

    def nonlocal_force(self, Psi, occ, col_block: int = 0):
        """F (n_atoms, 3) = nonlocal Hellmann-Feynman force; occ: (ns,) float64 CUDA tensor."""
        torch = _torch()
        pp, ld, ns = self._mat(Psi, "Psi")
        assert occ.is_cuda and occ.dtype == torch.float64 and occ.numel() == ns and occ.is_contiguous()
        F = torch.empty((max(self.n_atoms, 1), 3), dtype=torch.float64, device=Psi.device)
        ws = self._workspace(OP_NONLOCAL_FORCE, ns, col_block)
        _check(self.lib.sparc_gpu_nonlocal_force(self._ctx, pp, ld, ns, C.c_void_p(occ.data_ptr()),
                                                 C.c_void_p(F.data_ptr()), int(col_block), ws, self._stream()), "nonlocal_force")
        return F[:self.n_atoms]

    # ---- NEXT-1: subspace eigenproblem on the device ---------------------------------------------------
    def eigensolve(self, Hs, Ms):
        """Hs Z = Ms Z D on the device: returns (D (n,), Z (n, n) tensor holding the column-major matrix, info (2,) int32:
        status, sweeps).  Nothing is synchronised; read `info` after a stream sync."""
        torch = _torch()
        n = int(Hs.shape[0])
        assert Hs.is_cuda and Ms.is_cuda and Hs.shape == (n, n) and Ms.shape == (n, n) and Hs.is_contiguous() and Ms.is_contiguous()
        Z = torch.empty((n, n), dtype=torch.float64, device=Hs.device)
        D = torch.empty(n, dtype=torch.float64, device=Hs.device)
        info = torch.zeros(2, dtype=torch.int32, device=Hs.device)
        ws = self._workspace(OP_EIGENSOLVE, n, 0)
        _check(self.lib.sparc_gpu_eigensolve(self._ctx, n, C.c_void_p(Hs.data_ptr()), C.c_void_p(Ms.data_ptr()),
                                             C.c_void_p(Z.data_ptr()), C.c_void_p(D.data_ptr()), C.c_void_p(info.data_ptr()), ws,
                                             self._stream()), "eigensolve")
        return D, Z, info

    # ---- NEXT-4: complex (k-point) variant; complex matrices are torch.complex128 tensors (ncols, ld) ----------
    def set_kpoint(self, theta, supp_shift=None):
        th = (C.c_double * 3)(*[float(t) for t in theta])
        sh = None
        if supp_shift is not None:
            self._shift = np.ascontiguousarray(supp_shift, dtype=np.int8)
            sh = self._shift.ctypes.data
        _check(self.lib.sparc_gpu_set_kpoint(self._ctx, C.cast(th, C.c_void_p), sh), "set_kpoint")

    def _cmat(self, t, name: str):
        torch = _torch()
        if not (t.is_cuda and t.dtype == torch.complex128 and t.dim() == 2 and t.stride(1) == 1):
            raise ValueError(f"{name}: need a 2-D complex128 CUDA tensor (ncols, ld) contiguous along ld")
        if t.shape[1] < self.nd:
            raise ValueError(f"{name}: ld {t.shape[1]} < N_d {self.nd}")
        return C.c_void_p(t.data_ptr()), int(t.stride(0)) if t.shape[0] > 1 else int(t.shape[1]), int(t.shape[0])

    def hamiltonian_apply_k(self, X, Y=None):
        torch = _torch()
        xp, ldx, ncols = self._cmat(X, "X")
        if Y is None:
            Y = torch.empty_like(X)
        yp, ldy, _ = self._cmat(Y, "Y")
        ws = self._workspace(OP_HAMILTONIAN_APPLY_K, ncols, 0)
        _check(self.lib.sparc_gpu_hamiltonian_apply_k(self._ctx, xp, ldx, yp, ldy, ncols, ws, self._stream()), "hamiltonian_apply_k")
        return Y

    def chebyshev_filter_k(self, Psi, degree: int, a: float, b: float, a0: float, col_block: int = 0):
        pp, ld, ns = self._cmat(Psi, "Psi")
        ws = self._workspace(OP_CHEBYSHEV_FILTER_K, ns, col_block)
        _check(self.lib.sparc_gpu_chebyshev_filter_k(self._ctx, pp, ld, ns, int(degree), float(a), float(b), float(a0),
                                                     int(col_block), ws, self._stream()), "chebyshev_filter_k")
        return Psi

    def project_k(self, Psi, col_block: int = 0):
        torch = _torch()
        pp, ld, ns = self._cmat(Psi, "Psi")
        Hs = torch.empty((ns, ns), dtype=torch.complex128, device=Psi.device)
        Ms = torch.empty_like(Hs)
        ws = self._workspace(OP_PROJECT_K, ns, col_block)
        _check(self.lib.sparc_gpu_project_k(self._ctx, pp, ld, ns, C.c_void_p(Hs.data_ptr()), C.c_void_p(Ms.data_ptr()),
                                            int(col_block), ws, self._stream()), "project_k")
        return Hs, Ms       # element [j, i] = M_ij (column-major)

    def rotate_k(self, Psi, Q, row_panel: int = 0):
        torch = _torch()
        pp, ld, ns = self._cmat(Psi, "Psi")
        assert Q.is_cuda and Q.dtype == torch.complex128 and Q.shape == (ns, ns) and Q.is_contiguous()
        ws = self._workspace(OP_ROTATE_K, ns, row_panel)
        _check(self.lib.sparc_gpu_rotate_k(self._ctx, pp, ld, ns, C.c_void_p(Q.data_ptr()), int(row_panel), ws, self._stream()),
               "rotate_k")
        return Psi

    # ---- NEXT-2: local pieces of the row-partitioned projection / rotation (matrices (ncols, ld) with ld >= nrows) ------
    def gram(self, A, B, nrows: int, symmetric: bool = False, out=None):
        torch = _torch()
        m, n = int(A.shape[0]), int(B.shape[0])
        lda = int(A.stride(0)) if m > 1 else int(A.shape[1])
        ldb = int(B.stride(0)) if n > 1 else int(B.shape[1])
        Cm = out if out is not None else torch.empty((n, m), dtype=torch.float64, device=A.device)
        ws = self._workspace(OP_GRAM, max(m, n), 0)
        _check(self.lib.sparc_gpu_gram(self._ctx, C.c_void_p(A.data_ptr()), lda, C.c_void_p(B.data_ptr()), ldb, int(nrows), m, n,
                                       C.c_void_p(Cm.data_ptr()), 1 if symmetric else 0, ws, self._stream()), "gram")
        return Cm           # (n, m) tensor holding the column-major m x n matrix

    def rotate_rows(self, X, nrows: int, Q, row_panel: int = 0):
        ns = int(X.shape[0])
        ld = int(X.stride(0)) if ns > 1 else int(X.shape[1])
        ws = self._workspace(OP_ROTATE, ns, row_panel)
        _check(self.lib.sparc_gpu_rotate_rows(self._ctx, C.c_void_p(X.data_ptr()), ld, int(nrows), ns, C.c_void_p(Q.data_ptr()),
                                              int(row_panel), ws, self._stream()), "rotate_rows")
        return X

    def project(self, Psi, col_block: int = 0, Hs=None, Ms=None):
        torch = _torch()
        pp, ld, ns = self._mat(Psi, "Psi")
        if Hs is None:
            Hs = torch.empty((ns, ns), dtype=torch.float64, device=Psi.device)
        if Ms is None:
            Ms = torch.empty((ns, ns), dtype=torch.float64, device=Psi.device)
        ws = self._workspace(OP_PROJECT, ns, col_block)
        _check(self.lib.sparc_gpu_project(self._ctx, pp, ld, ns, C.c_void_p(Hs.data_ptr()),
                                          C.c_void_p(Ms.data_ptr()), int(col_block), ws, self._stream()), "project")
        return Hs, Ms       # (ns, ns) tensors holding the column-major matrices: element [j, i] = M_ij

    def rotate(self, Psi, Q, row_panel: int = 0):
        pp, ld, ns = self._mat(Psi, "Psi")
        assert Q.is_cuda and Q.shape == (ns, ns) and Q.is_contiguous()
        ws = self._workspace(OP_ROTATE, ns, row_panel)
        _check(self.lib.sparc_gpu_rotate(self._ctx, pp, ld, ns, C.c_void_p(Q.data_ptr()), int(row_panel), ws,
                                         self._stream()), "rotate")
        return Psi
