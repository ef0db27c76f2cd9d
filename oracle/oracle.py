"""ctypes/numpy wrapper of the CPU oracle (oracle/chefsi_oracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  The product package (paper_2302_09708_b200) never imports it, and this module never imports
the product's CUDA binding; the only shared module is the seeded input generator
``paper_2302_09708_b200.workloads`` (inputs only).

Two builds of the same source:
  liboracle_ld.so   acc_t = long double   (parity oracle)
  liboracle_f64.so  acc_t = double        (plain-FP64 CPU baseline that bench.py times)
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "chefsi_oracle.c")
_SRC_NEXT = os.path.join(_HERE, "chefsi_next_oracle.c")
_LOCK = threading.Lock()
_LIBS = {}


def build(force: bool = False) -> None:
    """Compile the oracle builds with gcc (-O3 -march=native -fopenmp): chefsi_oracle.c (the hot path) and
    chefsi_next_oracle.c, each with acc_t = long double and acc_t = double."""
    for src, stem in ((_SRC, "liboracle"), (_SRC_NEXT, "liboracle_next")):
        for tag, extra in (("ld", []), ("f64", ["-DORACLE_ACC_DOUBLE"])):
            out = os.path.join(_HERE, f"{stem}_{tag}.so")
            if (not force and os.path.exists(out)
                    and os.path.getmtime(out) >= os.path.getmtime(src)):
                continue
            cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                   "-fno-fast-math", *extra, src, "-o", out + ".tmp", "-lm"]
            subprocess.check_call(cmd)
            os.replace(out + ".tmp", out)


class _Ham(C.Structure):
    _fields_ = [("n", C.c_int32 * 3), ("h", C.c_double * 3), ("bc", C.c_int32 * 3),
                ("radius", C.c_int32), ("n_atoms", C.c_int32),
                ("supp_ptr", C.c_void_p), ("supp_idx", C.c_void_p), ("n_proj", C.c_void_p),
                ("chi_ptr", C.c_void_p), ("chi", C.c_void_p), ("gamma", C.c_void_p),
                ("veff", C.c_void_p)]


def _lib(acc: str = "ld"):
    with _LOCK:
        if acc not in _LIBS:
            build()
            lib = C.CDLL(os.path.join(_HERE, f"liboracle_{acc}.so"))
            P, I64, D = C.c_void_p, C.c_int64, C.c_double
            lib.oracle_acc_bits.restype = C.c_int
            lib.oracle_fd_weights.argtypes = [C.c_int, P]
            for name in ("oracle_laplacian", "oracle_vnl_apply", "oracle_h_apply"):
                getattr(lib, name).argtypes = [C.POINTER(_Ham), P, I64, P, I64, I64]
                getattr(lib, name).restype = None
            lib.oracle_chebyshev_filter.argtypes = [C.POINTER(_Ham), P, I64, I64, C.c_int, D, D, D]
            lib.oracle_chebyshev_filter.restype = C.c_int
            lib.oracle_gram.argtypes = [P, I64, P, I64, I64, P, I64, P, I64, P]
            lib.oracle_gram.restype = None
            lib.oracle_rotate.argtypes = [P, I64, I64, P, P, I64, P]
            lib.oracle_rotate.restype = None
            lib.oracle_project.argtypes = [C.POINTER(_Ham), P, I64, I64, P, P, P]
            lib.oracle_project.restype = None
            _LIBS[acc] = lib
        return _LIBS[acc]


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _fcols(x: np.ndarray) -> np.ndarray:
    x = np.asarray(x, dtype=np.float64)
    if x.ndim == 1:
        x = x.reshape(-1, 1)
    return np.asfortranarray(x)


class Hamiltonian:
    """Holds the (host) description of H for the oracle.  `wl` is a workloads.Workload-like object
    (attributes n, h, bc, fd_order, supp_ptr, supp_idx, n_proj, chi_ptr, chi, gamma, veff)."""

    def __init__(self, wl, acc: str = "ld", nonlocal_on: bool = True):
        self.lib = _lib(acc)
        self.nd = int(wl.n[0]) * int(wl.n[1]) * int(wl.n[2])
        self._keep = dict(
            supp_ptr=np.ascontiguousarray(wl.supp_ptr, dtype=np.int64),
            supp_idx=np.ascontiguousarray(wl.supp_idx, dtype=np.int32),
            n_proj=np.ascontiguousarray(wl.n_proj, dtype=np.int32),
            chi_ptr=np.ascontiguousarray(wl.chi_ptr, dtype=np.int64),
            chi=np.ascontiguousarray(wl.chi, dtype=np.float64),
            gamma=np.ascontiguousarray(wl.gamma, dtype=np.float64),
            veff=np.ascontiguousarray(wl.veff, dtype=np.float64))
        assert self._keep["veff"].shape[0] == self.nd
        h = _Ham()
        for k in range(3):
            h.n[k] = int(wl.n[k]); h.h[k] = float(wl.h[k]); h.bc[k] = int(wl.bc[k])
        h.radius = int(wl.fd_order) // 2
        h.n_atoms = int(self._keep["n_proj"].shape[0]) if nonlocal_on else 0
        for name in ("supp_ptr", "supp_idx", "n_proj", "chi_ptr", "chi", "gamma", "veff"):
            setattr(h, name, self._keep[name].ctypes.data)
        self.h = h

    def _apply(self, fn, X):
        X = _fcols(X)
        assert X.shape[0] == self.nd
        Y = np.empty_like(X, order="F")
        fn(C.byref(self.h), _ptr(X), X.shape[0], _ptr(Y), Y.shape[0], X.shape[1])
        return Y

    def laplacian(self, X):            # O2
        return self._apply(self.lib.oracle_laplacian, X)

    def vnl_apply(self, X):            # O4
        return self._apply(self.lib.oracle_vnl_apply, X)

    def apply(self, X):                # O5
        return self._apply(self.lib.oracle_h_apply, X)

    def chebyshev_filter(self, X, degree: int, a: float, b: float, a0: float):   # O6
        Y = _fcols(X).copy(order="F")
        rc = self.lib.oracle_chebyshev_filter(C.byref(self.h), _ptr(Y), Y.shape[0], Y.shape[1],
                                              int(degree), float(a), float(b), float(a0))
        if rc != 0:
            raise ValueError(f"oracle_chebyshev_filter: bad arguments (rc={rc})")
        return Y

    def project(self, Psi):            # O7 as one call (oracle_project: Y = H Psi, Hs = Psi^T Y, Ms = Psi^T Psi)
        Psi = _fcols(Psi)
        ns = Psi.shape[1]
        Y = np.empty_like(Psi, order="F")
        Hs = np.empty((ns, ns), dtype=np.float64, order="F")
        Ms = np.empty((ns, ns), dtype=np.float64, order="F")
        self.lib.oracle_project(C.byref(self.h), _ptr(Psi), Psi.shape[0], ns, _ptr(Y), _ptr(Hs), _ptr(Ms))
        return Hs, Ms


def fd_weights(radius: int) -> np.ndarray:   # O1
    w = np.zeros(radius + 1)
    _lib("ld").oracle_fd_weights(int(radius), _ptr(w))
    return w


def gram(A, B, I: Optional[Sequence[int]] = None, J: Optional[Sequence[int]] = None, lib=None,
         acc: str = "ld") -> np.ndarray:
    """out[i,j] = sum_r A[r, I[i]] B[r, J[j]]   (O7)."""
    lib = lib or _lib(acc)
    A, B = _fcols(A), _fcols(B)
    assert A.shape[0] == B.shape[0]
    Ia = None if I is None else np.ascontiguousarray(I, dtype=np.int64)
    Ja = None if J is None else np.ascontiguousarray(J, dtype=np.int64)
    nI = A.shape[1] if Ia is None else Ia.shape[0]
    nJ = B.shape[1] if Ja is None else Ja.shape[0]
    out = np.empty((nI, nJ), dtype=np.float64, order="F")
    lib.oracle_gram(_ptr(A), A.shape[0], _ptr(B), B.shape[0], A.shape[0], _ptr(Ia), nI, _ptr(Ja), nJ,
                    _ptr(out))
    return out


def rotate(Psi, Q, rows: Optional[Sequence[int]] = None, acc: str = "ld") -> np.ndarray:
    """out[k,:] = Psi[rows[k],:] @ Q   (O8)."""
    lib = _lib(acc)
    Psi, Q = _fcols(Psi), _fcols(Q)
    ns = Psi.shape[1]
    assert Q.shape == (ns, ns)
    R = None if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    nrows = Psi.shape[0] if R is None else R.shape[0]
    out = np.empty((nrows, ns), dtype=np.float64, order="F")
    lib.oracle_rotate(_ptr(Psi), Psi.shape[0], ns, _ptr(Q), _ptr(R), nrows, _ptr(out))
    return out


# ======================================================================================================================
# SURVEY.md section 8(f) "next" rows (oracle/chefsi_next_oracle.c)
# ======================================================================================================================
_NLIBS = {}


class _HamK(C.Structure):
    _fields_ = [("base", _Ham), ("theta", C.c_double * 3), ("shift", C.c_void_p)]


def _nlib(acc: str = "ld"):
    with _LOCK:
        if acc not in _NLIBS:
            build()
            lib = C.CDLL(os.path.join(_HERE, f"liboracle_next_{acc}.so"))
            P, I64, D, I = C.c_void_p, C.c_int64, C.c_double, C.c_int
            lib.oracle_fd1_weights.argtypes = [I, P]
            lib.oracle_gradient.argtypes = [C.POINTER(_Ham), I, P, I64, P, I64, I64]
            lib.oracle_gradient.restype = None
            lib.oracle_nl_project.argtypes = [C.POINTER(_Ham), P, I64, I64, P]
            lib.oracle_nl_project.restype = None
            lib.oracle_nonlocal_force.argtypes = [C.POINTER(_Ham), P, I64, I64, P, P, P]
            lib.oracle_nonlocal_force.restype = None
            lib.oracle_sygv.argtypes = [I64, P, P, P, P]
            lib.oracle_sygv.restype = I
            lib.oracle_h_apply_k.argtypes = [C.POINTER(_HamK), P, I64, P, I64, I64]
            lib.oracle_h_apply_k.restype = None
            lib.oracle_chebyshev_filter_k.argtypes = [C.POINTER(_HamK), P, I64, I64, I, D, D, D]
            lib.oracle_chebyshev_filter_k.restype = I
            lib.oracle_gram_k.argtypes = [P, I64, P, I64, I64, I64, I64, P]
            lib.oracle_gram_k.restype = None
            lib.oracle_rotate_k.argtypes = [P, I64, I64, I64, P, P]
            lib.oracle_rotate_k.restype = None
            _NLIBS[acc] = lib
        return _NLIBS[acc]


def fd1_weights(radius: int) -> np.ndarray:        # G1
    w = np.zeros(radius + 1)
    _nlib("ld").oracle_fd1_weights(int(radius), _ptr(w))
    return w


class Forces:
    """Gradient stencil, projector contraction and nonlocal force of the oracle (G2-G4) for a Workload-like `wl`."""

    def __init__(self, wl, acc: str = "ld"):
        self._H = Hamiltonian(wl, acc="ld")              # only for its packed descriptor
        self.h = self._H.h
        self.lib = _nlib(acc)
        self.nd = self._H.nd
        self.n_proj_total = int(np.sum(wl.n_proj))
        self.n_atoms = int(len(wl.n_proj))

    def gradient(self, X, axis: int):
        X = _fcols(X)
        Y = np.empty_like(X, order="F")
        self.lib.oracle_gradient(C.byref(self.h), int(axis), _ptr(X), X.shape[0], _ptr(Y), Y.shape[0], X.shape[1])
        return Y

    def nl_project(self, X):
        X = _fcols(X)
        W = np.empty((max(self.n_proj_total, 1), X.shape[1]), dtype=np.float64, order="F")
        self.lib.oracle_nl_project(C.byref(self.h), _ptr(X), X.shape[0], X.shape[1], _ptr(W))
        return W[:self.n_proj_total]

    def nonlocal_force(self, Psi, occ):
        Psi = _fcols(Psi)
        occ = np.ascontiguousarray(occ, dtype=np.float64)
        assert occ.shape[0] == Psi.shape[1]
        F = np.zeros((max(self.n_atoms, 1), 3), dtype=np.float64)
        scratch = np.empty_like(Psi, order="F")
        self.lib.oracle_nonlocal_force(C.byref(self.h), _ptr(Psi), Psi.shape[0], Psi.shape[1], _ptr(occ), _ptr(F),
                                       _ptr(scratch))
        return F[:self.n_atoms]


def sygv(Hs, Ms, acc: str = "ld"):
    """Generalized symmetric-definite eigenproblem Hs Z = Ms Z D (E1-E4): returns (D ascending, Z with Z^T Ms Z = I)."""
    Hs, Ms = _fcols(Hs), _fcols(Ms)
    n = Hs.shape[0]
    assert Hs.shape == (n, n) and Ms.shape == (n, n)
    Z = np.zeros((n, n), dtype=np.float64, order="F")
    D = np.zeros(n, dtype=np.float64)
    rc = _nlib(acc).oracle_sygv(n, _ptr(Hs), _ptr(Ms), _ptr(Z), _ptr(D))
    if rc != 0:
        raise ValueError(f"oracle_sygv failed (rc={rc}: 1 = Ms not positive definite, 2 = Jacobi did not converge)")
    return D, Z


def _cplx(x):
    x = np.asarray(x, dtype=np.complex128)
    if x.ndim == 1:
        x = x.reshape(-1, 1)
    return np.asfortranarray(x)


class HamiltonianK:
    """Complex (k-point) operator of the oracle (K1-K4).  `theta`: Bloch phase k_a L_a per axis; `wl.supp_shift`
    ([supp_total, 3] int8 image shifts of the support rows) is taken when present."""

    def __init__(self, wl, theta, acc: str = "ld"):
        self._H = Hamiltonian(wl, acc="ld")
        self.lib = _nlib(acc)
        self.nd = self._H.nd
        hk = _HamK()
        hk.base = self._H.h
        for a in range(3):
            hk.theta[a] = float(theta[a]) if int(wl.bc[a]) == 0 else 0.0
        sh = getattr(wl, "supp_shift", None)
        self._shift = None if sh is None else np.ascontiguousarray(sh, dtype=np.int8)
        hk.shift = None if self._shift is None else self._shift.ctypes.data
        self.hk = hk

    def apply(self, X):
        X = _cplx(X)
        Y = np.empty_like(X, order="F")
        self.lib.oracle_h_apply_k(C.byref(self.hk), _ptr(X), X.shape[0], _ptr(Y), Y.shape[0], X.shape[1])
        return Y

    def chebyshev_filter(self, X, degree, a, b, a0):
        Y = _cplx(X).copy(order="F")
        rc = self.lib.oracle_chebyshev_filter_k(C.byref(self.hk), _ptr(Y), Y.shape[0], Y.shape[1], int(degree),
                                                float(a), float(b), float(a0))
        if rc != 0:
            raise ValueError("oracle_chebyshev_filter_k: bad arguments")
        return Y


def gram_k(A, B, acc: str = "ld"):
    A, B = _cplx(A), _cplx(B)
    out = np.empty((A.shape[1], B.shape[1]), dtype=np.complex128, order="F")
    _nlib(acc).oracle_gram_k(_ptr(A), A.shape[0], _ptr(B), B.shape[0], A.shape[0], A.shape[1], B.shape[1], _ptr(out))
    return out


def rotate_k(Psi, Q, acc: str = "ld"):
    Psi, Q = _cplx(Psi), _cplx(Q)
    out = np.empty_like(Psi, order="F")
    _nlib(acc).oracle_rotate_k(_ptr(Psi), Psi.shape[0], Psi.shape[0], Psi.shape[1], _ptr(Q), _ptr(out))
    return out
