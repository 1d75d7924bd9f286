"""msolve_spmv_csr_noalloc (include/msolve.h, csrc/noalloc.cu): the SpMV + fused <x, A x> of Alg. 1 l.18-19 for callers
that cannot allocate device memory -- no handle, scratch in a static device array -- against the existing path
(msolve_create_csr + msolve_spmv) on the same inputs, on calls in a row that share that array.

Collected last on purpose (the suite runs with pytest -x); needs nothing from the tests before it."""
import ctypes

import numpy as np
import pytest
import torch

from paper_1102_2143_b200 import workloads as W

pytestmark = pytest.mark.gpu

# the bars of tests/test_gpu_lattice.py::test_lattice_spmv_matches_oracle for one SpMV and its dot product
EPS = {np.complex128: 1e-13, np.complex64: 1e-5, np.float64: 1e-13, np.float32: 1e-5}


@pytest.fixture(scope="module")
def ms():
    from paper_1102_2143_b200 import binding, build
    build.build()
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _cases(dtype):
    """(rowptr, colidx, val) of three matrices of different sizes: a later, smaller call finds the partials of an
    earlier, larger one in the shared scratch array."""
    real = dtype in (np.float64, np.float32)
    out = []
    for w in (W.config2(), W.config5(n=(1 << 14) + 13), W.config1()):
        val = w.val.real if real else w.val
        out.append((w.rowptr, w.colidx, np.ascontiguousarray(val).astype(dtype)))
    return out


def _existing_path(ms, rowptr, colidx, val, x):
    A = ms.msolve_create_csr(dev(rowptr), dev(colidx), dev(val))
    y, dot = ms.msolve_spmv(A, dev(x))
    y = y.cpu().numpy()
    ms.msolve_destroy(A)
    return y, dot


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64, np.float64, np.float32])
def test_noalloc_matches_existing_path_on_calls_in_a_row(ms, dtype):
    rng = np.random.default_rng(11)
    real = dtype in (np.float64, np.float32)
    eps = EPS[dtype]
    dot_buf = torch.empty(2, dtype=torch.float64, device="cuda")
    for rowptr, colidx, val in _cases(dtype):
        n = rowptr.size - 1
        d_rowptr, d_colidx, d_val = dev(rowptr), dev(colidx), dev(val)
        for call in range(2):                                   # two calls in a row on the same matrix, different x
            x = rng.standard_normal(n) if real else rng.standard_normal(n) + 1j * rng.standard_normal(n)
            x = x.astype(dtype)
            y_ref, dot_ref = _existing_path(ms, rowptr, colidx, val, x)
            y_buf = torch.full((n,), float("nan"), dtype=d_val.dtype, device="cuda")
            dot_buf.fill_(float("nan"))
            y, dot = ms.msolve_spmv_csr_noalloc(d_rowptr, d_colidx, d_val, dev(x), y=y_buf, dot=dot_buf)
            assert y.data_ptr() == y_buf.data_ptr() and dot.data_ptr() == dot_buf.data_ptr()
            torch.cuda.synchronize()
            y = y.cpu().numpy()
            d = dot.cpu().numpy()
            assert np.linalg.norm(y - y_ref) <= eps * np.linalg.norm(y_ref), (n, call)
            assert abs(complex(d[0], d[1]) - dot_ref) <= eps * abs(dot_ref), (n, call)
            if real:
                assert d[1] == 0.0
            # the same call again: same bytes (fixed-order reduction), whatever the scratch array held before
            y2, dot2 = ms.msolve_spmv_csr_noalloc(d_rowptr, d_colidx, d_val, dev(x))
            torch.cuda.synchronize()
            assert np.array_equal(y2.cpu().numpy(), y) and np.array_equal(dot2.cpu().numpy(), d)


def test_noalloc_empty_system_and_limits(ms):
    lib = ms.load_library()
    # n = 0: the dot product is written (zero), nothing else is touched
    dot = torch.full((2,), 7.0, dtype=torch.float64, device="cuda")
    rowptr = torch.zeros(1, dtype=torch.int32, device="cuda")
    empty = torch.empty(0, dtype=torch.complex128, device="cuda")
    ms.msolve_spmv_csr_noalloc(rowptr, torch.empty(0, dtype=torch.int32, device="cuda"), empty, empty, dot=dot)
    torch.cuda.synchronize()
    assert dot.cpu().tolist() == [0.0, 0.0]
    # beyond the static scratch: rejected before anything is launched, with the limit in the message
    p = ctypes.c_void_p(rowptr.data_ptr())
    rc = lib.msolve_spmv_csr_noalloc(ms.MSOLVE_NOALLOC_MAX_ROWS + 1, p, p, p, ms.MSOLVE_C128, p, p, ctypes.c_void_p(dot.data_ptr()), None)
    assert rc == -1 and b"MSOLVE_NOALLOC_MAX_ROWS" in lib.msolve_last_error()
    assert lib.msolve_spmv_csr_noalloc(-1, p, p, p, ms.MSOLVE_C128, p, p, ctypes.c_void_p(dot.data_ptr()), None) == -1
    assert lib.msolve_spmv_csr_noalloc(4, p, p, p, 9, p, p, ctypes.c_void_p(dot.data_ptr()), None) == -1
    assert lib.msolve_spmv_csr_noalloc(4, p, p, p, ms.MSOLVE_C128, p, p, None, None) == -1
    torch.cuda.synchronize()
    assert dot.cpu().tolist() == [0.0, 0.0]


def test_noalloc_at_the_maximum_size(ms):
    # n = MSOLVE_NOALLOC_MAX_ROWS exactly: every entry of the scratch array is used (tridiagonal real matrix, fp64)
    n = ms.MSOLVE_NOALLOC_MAX_ROWS
    i = np.arange(n)
    counts = np.full(n, 3, dtype=np.int64)
    counts[0] = counts[-1] = 2
    rowptr = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    cols = np.stack([i - 1, i, i + 1], axis=1).ravel()
    keep = (cols >= 0) & (cols < n)
    colidx = cols[keep].astype(np.int32)
    val = np.tile(np.array([-1.0, 2.5, -1.0]), n)[keep]
    x = np.random.default_rng(3).standard_normal(n)
    y_ref = 2.5 * x
    y_ref[1:] -= x[:-1]
    y_ref[:-1] -= x[1:]
    y, dot = ms.msolve_spmv_csr_noalloc(dev(rowptr), dev(colidx), dev(val), dev(x))
    torch.cuda.synchronize()
    assert np.linalg.norm(y.cpu().numpy() - y_ref) <= 1e-13 * np.linalg.norm(y_ref)
    d = dot.cpu().numpy()
    assert abs(d[0] - np.dot(x, y_ref)) <= 1e-12 * abs(np.dot(x, y_ref)) and d[1] == 0.0
