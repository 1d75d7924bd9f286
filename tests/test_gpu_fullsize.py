"""Full-size parity in the launch configuration bench.py times (BASELINE configs[3] and [4]).

config 4 (32^3x64, N = 6.29 M, c128, BSR3, 16 shifts): the oracle runs the whole solve on the host
(about a minute) and every solution is compared element by element; true residuals are checked
on sampled rows computed one by one in numpy.  config 5 (N = 2^22, 134 M nnz, 32 shifts) is run
on the GPU at full size and checked through size-independent properties (sampled true residual
rows, status, monotone conv_iter) plus a bounded oracle comparison at a fixed iteration count.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1102_2143_b200 import workloads as W

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def sampled_true_residual(w, x, sigma, rows):
    """(b - (A + sigma) x)_i for sampled rows i, straight from the CSR arrays (numpy, fp64)."""
    out = np.empty(rows.size, dtype=np.complex128)
    for t, i in enumerate(rows):
        lo, hi = w.rowptr[i], w.rowptr[i + 1]
        out[t] = w.b[i] - (np.dot(w.val[lo:hi], x[w.colidx[lo:hi]]) + sigma * x[i])
    return out


@pytest.fixture(scope="module")
def ms():
    from paper_1102_2143_b200 import binding, build
    build.build()
    return binding


def test_config4_full_c128_bsr3_vs_oracle(ms):
    w = W.config4()
    A = ms.msolve_create_bsr3(dev(w.browptr), dev(w.bcolidx), dev(w.blocks))
    res = ms.msolve_cgm(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    x = res.x.cpu().numpy()
    ref = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, w.tol, w.max_iter)
    assert res.status == ref.status == 0
    assert abs(res.iterations - ref.iterations) <= 2
    assert np.all(np.abs(res.conv_iter - ref.conv_iter) <= 2)
    rows = np.random.default_rng(0).integers(0, w.n, 4000)
    for k, s in enumerate(w.shifts):
        d = np.linalg.norm(x[k] - ref.x[k]) / np.linalg.norm(ref.x[k])
        assert d <= 1e-9, (k, d)
        rs = sampled_true_residual(w, x[k], s, rows)
        # ||b|| = 1: an rms residual entry of tol/sqrt(n) corresponds to ||r|| = tol
        assert np.sqrt(np.mean(np.abs(rs) ** 2) * w.n) <= 10 * w.tol, k
    ms.msolve_destroy(A)
    del res, x
    # the same matrix as CSR (AUTO = TMA-staged vector-CSR kernel), element by element
    A = ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val))
    rc = ms.msolve_cgm(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    assert rc.status == 0 and abs(rc.iterations - ref.iterations) <= 2
    assert np.all(np.abs(rc.conv_iter - ref.conv_iter) <= 2)
    xc = rc.x.cpu().numpy()
    for k in range(len(w.shifts)):
        d = np.linalg.norm(xc[k] - ref.x[k]) / np.linalg.norm(ref.x[k])
        assert d <= 1e-9, (k, d)
    ms.msolve_destroy(A)
    del rc, xc
    torch.cuda.empty_cache()
    # complex64 data path at full size: properties only
    A = ms.msolve_create_bsr3(dev(w.browptr), dev(w.bcolidx), dev(w.blocks.astype(np.complex64)))
    r32 = ms.msolve_cgm(A, dev(w.b.astype(np.complex64)), w.shifts, 1e-5, w.max_iter)
    assert r32.status == 0 and abs(r32.iterations - 12) <= 2
    x32 = r32.x.cpu().numpy()
    for k in (0, 8, 15):
        d = np.linalg.norm(x32[k].astype(np.complex128) - ref.x[k]) / np.linalg.norm(ref.x[k])
        assert d <= 1e-4, (k, d)       # c64 at tol 1e-5 against the converged c128 oracle
    ms.msolve_destroy(A)


def test_config5_full_properties_and_bounded_oracle(ms):
    w = W.config5()
    for dtype, tol in ((np.complex64, 1e-5), (np.complex128, 1e-10)):
        A = ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val.astype(dtype)))
        b = dev(w.b.astype(dtype))
        res = ms.msolve_cgm(A, b, w.shifts, tol, w.max_iter)
        assert res.status == 0
        assert np.all(np.diff(res.conv_iter) <= 0) and res.iterations == res.conv_iter.max()
        rows = np.random.default_rng(1).integers(0, w.n, 2000)
        for k in (0, 13, 31):
            xk = res.x[k].cpu().numpy().astype(np.complex128)
            rs = sampled_true_residual(w, xk, w.shifts[k], rows)
            assert np.sqrt(np.mean(np.abs(rs) ** 2) * w.n) <= 10 * tol, (dtype, k)
        if dtype == np.complex128:
            # bounded oracle comparison: iterate after 3 iterations, 3 shifts
            sh = w.shifts[[0, 13, 31]]
            g = ms.msolve_cgm(A, b, sh, 0.0, 3)
            o = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, sh, 0.0, 3)
            gx = g.x.cpu().numpy()
            for k in range(3):
                assert np.linalg.norm(gx[k] - o.x[k]) / np.linalg.norm(o.x[k]) <= 1e-12
            assert np.allclose(g.relres, o.relres, rtol=1e-9)
        ms.msolve_destroy(A)
        del A, b, res
        torch.cuda.empty_cache()
