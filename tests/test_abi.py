"""CPU-side checks of the C-ABI boundary: the library builds, loads, exports every symbol that
include/sparc_gpu.h declares, and its host-side validation answers with the documented status codes.
No kernel is launched here (there is no GPU in the CPU container)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2302_09708_b200 import api, workloads as wlmod

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    return api.load_library()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "sparc_gpu.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sparc_gpu_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    syms = declared_symbols()
    assert len(syms) >= 13
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in include/sparc_gpu.h but not exported"
    assert sorted(api.EXPORTS) == syms


def test_version_and_error_strings(lib):
    assert b"sm_100a" in lib.sparc_gpu_version()
    seen = set()
    for code in range(0, -8, -1):
        msg = lib.sparc_gpu_error_string(code)
        assert msg and msg != b"unknown status"
        seen.add(msg)
    assert len(seen) == 8
    assert lib.sparc_gpu_error_string(-99) == b"unknown status"


def _desc(wl, **over):
    keep = dict(supp_ptr=np.ascontiguousarray(wl.supp_ptr, np.int64),
                supp_idx=np.ascontiguousarray(wl.supp_idx, np.int32),
                n_proj=np.ascontiguousarray(wl.n_proj, np.int32),
                chi_ptr=np.ascontiguousarray(wl.chi_ptr, np.int64),
                chi=np.ascontiguousarray(wl.chi, np.float64),
                gamma=np.ascontiguousarray(wl.gamma, np.float64),
                veff=np.ascontiguousarray(wl.veff, np.float64))
    keep.update({k: v for k, v in over.items() if k in keep})
    d = api.Desc()
    for k in range(3):
        d.n[k], d.h[k], d.bc[k] = int(wl.n[k]), float(wl.h[k]), int(wl.bc[k])
    d.fd_order = over.get("fd_order", wl.fd_order)
    d.n_atoms = wl.n_atoms
    for name, arr in keep.items():
        setattr(d, name, arr.ctypes.data)
    d.device = 0
    return d, keep


def test_descriptor_validation_without_gpu(lib):
    wl = wlmod.make_workload(0)
    ctx = C.c_void_p()
    assert lib.sparc_gpu_create(None, C.byref(ctx)) == -1
    d, keep = _desc(wl, fd_order=13)
    assert lib.sparc_gpu_create(C.byref(d), C.byref(ctx)) == -2          # odd order
    d, keep = _desc(wl, fd_order=14)
    assert lib.sparc_gpu_create(C.byref(d), C.byref(ctx)) == -2          # radius > 6
    bad = wl.supp_idx.copy()
    bad[3], bad[4] = bad[4], bad[3]
    d, keep = _desc(wl, supp_idx=bad)
    assert lib.sparc_gpu_create(C.byref(d), C.byref(ctx)) == -4          # not ascending
    bad = wl.supp_idx.copy()
    bad[0] = wl.nd
    d, keep = _desc(wl, supp_idx=bad)
    assert lib.sparc_gpu_create(C.byref(d), C.byref(ctx)) == -4          # out of range
    badp = wl.chi_ptr.copy()
    badp[-1] += 1
    d, keep = _desc(wl, chi_ptr=badp)
    assert lib.sparc_gpu_create(C.byref(d), C.byref(ctx)) == -4
    # periodic axis shorter than the stencil (R10)
    small = wlmod.make_custom("s", (12, 16, 16), (0.5,) * 3, (1, 0, 0), 1, 1, np.zeros((0, 3)), [], 2.0)
    d, keep = _desc(small)
    d.bc[0] = 0
    assert lib.sparc_gpu_create(C.byref(d), C.byref(ctx)) == -2
    # a valid descriptor: without an sm_100 device the answer is UNSUPPORTED, never a CPU fallback
    import torch
    if not torch.cuda.is_available():
        d, keep = _desc(wl)
        assert lib.sparc_gpu_create(C.byref(d), C.byref(ctx)) == -2
        assert not ctx.value
        with pytest.raises(RuntimeError):
            api.SparcGpu(wl)


def test_null_context_calls_are_rejected(lib):
    out = C.c_int64()
    assert lib.sparc_gpu_workspace_bytes(None, 0, 4, 0, C.byref(out)) == -1
    assert lib.sparc_gpu_hamiltonian_apply(None, None, 0, None, 0, 1, None, None) == -1
    assert lib.sparc_gpu_chebyshev_filter(None, None, 0, 1, 2, 0.0, 1.0, -1.0, 0, None, None) == -1
    assert lib.sparc_gpu_project(None, None, 0, 1, None, None, 0, None, None) == -1
    assert lib.sparc_gpu_rotate(None, None, 0, 1, None, 0, None, None) == -1
    assert lib.sparc_gpu_destroy(None) == -1
    assert lib.sparc_gpu_set_option(None, b"nonlocal", 0) == -1
