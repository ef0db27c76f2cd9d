"""sparc_gpu_gram_static, the one entry point of the library that allocates nothing.

Who needs it: a caller that cannot get device memory at the moment it wants X^T Y -- an SCF driver whose own arena already
holds all of HBM (or that runs under a per-process cap), code in the middle of an overlapped multi-stream region that a
cudaMalloc / cudaFree would stall, a plug-in whose host application owns the allocator.  Such a caller has no context
(sparc_gpu_create uploads tables) and no workspace to lend, so the split-K partial products of this variant live in a
16 MiB array compiled into the library, one per GPU, shared by all calls and never cleared.

What is checked: the new entry point against the existing path (sparc_gpu_gram with a caller-owned workspace) at the
tolerance the Gram tests use (1e-13 in the Frobenius norm; where both paths take the same row split the results must be
bit-identical), on TWO calls in a row whose shapes differ, so that whatever the first call left in the shared array would
show up in the second; the size limit; the argument errors.  The file is named so that pytest collects it last (a failure
here under `-x` hides no other test) and it builds its own inputs, so it passes alone in a fresh process as well as
after the rest of the suite."""
import ctypes as C

import numpy as np
import pytest

from paper_2302_09708_b200 import workloads as wlmod

pytestmark = pytest.mark.gpu

TOL = 1e-13          # the gate of tests/test_gpu_dist.py::test_gram_and_rotate_rows_entry_points


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


@pytest.fixture(scope="module")
def api():
    from paper_2302_09708_b200 import api as a
    return a


def fro(G, O):
    return float(np.linalg.norm(G - O) / np.linalg.norm(O))


def _block(api, torch, rows, cols, ld, stream_id):
    """rows x cols column-major block with leading dimension ld, filled on the device by the workloads' generator."""
    t = torch.zeros((cols, ld), dtype=torch.float64, device="cuda:0")
    api.fill_uniform(t, 20230209, stream_id, 0, -1.0, 1.0)
    return t


def test_gram_static_matches_gram_on_two_calls_in_a_row(torch, api):
    g = api.SparcGpu(wlmod.make_workload(0))          # only the EXISTING path needs a context and a workspace
    try:
        # call 1: tall block, small output (many row splits: the shared array is filled with partials), odd sizes, unaligned ld
        # call 2: a different, larger output right after it, symmetric (upper tiles + mirror), aligned ld
        # call 3: the first shape again, after the array has been overwritten by call 2
        cases = [dict(nr=70001, m=37, n=21, lda=70001, ldb=70004, sym=False),
                 dict(nr=40960, m=300, n=300, lda=40960, ldb=40960, sym=True),
                 dict(nr=70001, m=37, n=21, lda=70001, ldb=70004, sym=False)]
        blocks, results = [], []
        for k, c in enumerate(cases):
            A = _block(api, torch, c["nr"], c["m"], c["lda"], 101 + (k % 2))
            B = A if c["sym"] else _block(api, torch, c["nr"], c["n"], c["ldb"], 201 + (k % 2))
            blocks.append((A, B))
        for c, (A, B) in zip(cases, blocks):           # the calls under test, back to back on one stream, nothing in between
            results.append(api.gram_static(A, B, c["nr"], symmetric=c["sym"]))
        torch.cuda.synchronize()
        for k, (c, (A, B)) in enumerate(zip(cases, blocks)):
            ref = api.colmajor_to_numpy(g.gram(A, B, c["nr"], symmetric=c["sym"]))
            got = api.colmajor_to_numpy(results[k])
            assert got.shape == (c["m"], c["n"]) and np.isfinite(got).all()
            err = fro(got, ref)
            print(f"[no-alloc] gram_static vs gram, call {k + 1} ({c['nr']} x {c['m']} x {c['n']}, symmetric {c['sym']}): {err:.2e}")
            assert err <= TOL
            if c["sym"]:
                assert np.array_equal(got, got.T)
            if 64 * c["m"] * c["n"] <= api.GRAM_STATIC_MAX_ELEMS:      # same cap on the partials => same row split => same bits
                assert np.array_equal(got, ref)
            # and against a plain float64 product on the host, so that the two paths cannot be wrong together
            Ah, Bh = api.colmajor_to_numpy(A, c["nr"]), api.colmajor_to_numpy(B, c["nr"])
            assert fro(got, Ah.T @ Bh) <= 1e-12
        assert np.array_equal(api.colmajor_to_numpy(results[0]), api.colmajor_to_numpy(results[2]))   # repeatable
    finally:
        g.close()


def test_gram_static_limit_and_argument_errors(torch, api):
    lib = api.load_library()
    assert api.GRAM_STATIC_MAX_ELEMS == 2097152
    nr = 64
    A = torch.zeros((1449, nr), dtype=torch.float64, device="cuda:0")
    out = torch.full((1449 * 1449,), 7.0, dtype=torch.float64, device="cuda:0")
    # 1448 x 1448 = 2 096 704 fits, 1449 x 1449 = 2 099 601 does not: clear status, C untouched
    api.gram_static(A[:1448], A[:1448], nr, out=out[:1448 * 1448].view(1448, 1448))
    torch.cuda.synchronize()
    assert float(out[:1448 * 1448].abs().max()) == 0.0
    with pytest.raises(api.SparcGpuError) as ei:
        api.gram_static(A, A, nr, out=out.view(1449, 1449))
    assert ei.value.code == -8 and "static scratch" in str(ei.value)
    torch.cuda.synchronize()
    assert float(out[-1]) == 7.0
    # nrows = 0: C = 0 without touching A, B
    z = torch.full((3, 2), 5.0, dtype=torch.float64, device="cuda:0")
    null, s = C.c_void_p(0), C.c_void_p(torch.cuda.current_stream().cuda_stream)
    assert lib.sparc_gpu_gram_static(0, null, 0, null, 0, 0, 2, 3, C.c_void_p(z.data_ptr()), 0, s) == 0
    torch.cuda.synchronize()
    assert float(z.abs().max()) == 0.0
    p = C.c_void_p(A.data_ptr())
    assert lib.sparc_gpu_gram_static(0, p, nr, p, nr, nr, 2, 3, C.c_void_p(z.data_ptr()), 1, s) == -1    # symmetric, m != n
    assert lib.sparc_gpu_gram_static(0, p, nr - 1, p, nr, nr, 2, 3, C.c_void_p(z.data_ptr()), 0, s) == -1   # lda < nrows
    assert lib.sparc_gpu_gram_static(0, null, nr, p, nr, nr, 2, 3, C.c_void_p(z.data_ptr()), 0, s) == -1    # NULL A
    assert lib.sparc_gpu_gram_static(-1, p, nr, p, nr, nr, 2, 3, C.c_void_p(z.data_ptr()), 0, s) == -1      # bad device
    assert lib.sparc_gpu_gram_static(0, p, nr, p, nr, nr, 0, 3, null, 0, s) == 0                            # empty output
