"""Row partition on one device (msolve_slabs_*, csrc/slab.cu): P slabs of one matrix, halo
exchange of the gathered vector before every SpMV, dot products summed over the slabs.  Against the oracle on the
UNPARTITIONED matrix with the usual bars, for every P; across P the solutions agree to rounding (the dot products
are grouped by slab), and a repeated solve returns the same bytes."""
import numpy as np
import pytest
import scipy.sparse as sp
import torch

import oracle
from paper_1102_2143_b200 import workloads as W
from test_gpu_parity import MAXABS_C, REL, dev, ms  # noqa: F401

pytestmark = pytest.mark.gpu


def make_slabs(ms, w, dtype, fmt, nslabs, flags=0):
    if fmt == "bsr3":
        return ms.msolve_slabs_create_bsr3(w.browptr, w.bcolidx, w.blocks.astype(dtype), nslabs, flags=flags)
    return ms.msolve_slabs_create_csr(w.rowptr, w.colidx, w.val.astype(dtype), nslabs, flags=flags)


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("fmt", ["csr", "bsr3"])
@pytest.mark.parametrize("nslabs", [1, 2, 3, 8])
def test_slab_spmv_matches_oracle(ms, nslabs, fmt, dtype):
    w = W.config2(extents=(6, 4, 5, 8))
    rng = np.random.default_rng(7)
    x = (rng.standard_normal(w.n) + 1j * rng.standard_normal(w.n)).astype(dtype)
    S = make_slabs(ms, w, dtype, fmt, nslabs)
    y, dot = ms.msolve_slabs_spmv(S, dev(x))
    ref = oracle.spmv(w.rowptr, w.colidx, w.val.astype(dtype), x)
    eps = 1e-13 if dtype == np.complex128 else 1e-5
    assert np.linalg.norm(y.cpu().numpy() - ref) / np.linalg.norm(ref) < eps
    ref_dot = np.vdot(x.astype(np.complex128), ref.astype(np.complex128))
    assert abs(dot - ref_dot) / abs(ref_dot) < eps
    halo = ms.msolve_slabs_halo_elements(S)
    assert len(halo) == nslabs and (nslabs == 1) == (sum(halo) == 0)
    ms.msolve_slabs_destroy(S)


def _check(w, dtype, tol, g, o):
    assert g.status == o.status == 0 and abs(g.iterations - o.iterations) <= 2
    assert np.all(np.abs(g.conv_iter - o.conv_iter) <= 2)
    A = sp.csr_matrix((w.val, w.colidx, w.rowptr), shape=(w.n, w.n))
    x = g.x.cpu().numpy()
    for k, s in enumerate(w.shifts):
        diff = x[k].astype(np.complex128) - o.x[k].astype(np.complex128)
        assert np.linalg.norm(diff) <= REL[dtype] * np.linalg.norm(o.x[k]), k
        assert np.abs(diff).max() <= MAXABS_C * REL[dtype] * np.abs(o.x[k]).max(), k
        xk = x[k].astype(np.complex128)
        assert np.linalg.norm(w.b - (A @ xk + s * xk)) <= 10 * tol * np.linalg.norm(w.b), k
        assert g.relres[k] <= tol * (1 + 1e-12)
    return x


@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
@pytest.mark.parametrize("which,fmt", [("c2", "csr"), ("c2", "bsr3"), ("c4s", "bsr3"), ("c4s", "csr"), ("c5", "csr")])
def test_slabs_cgm_matches_oracle_for_every_p(ms, which, fmt, dtype, tol):
    w = {"c2": W.config2, "c4s": lambda: W.config4(extents=(8, 8, 8, 16), want_csr=True),
         "c5": lambda: W.config5(n=(1 << 15) + 36)}[which]()
    o = oracle.cgm(w.rowptr, w.colidx, w.val.astype(dtype), w.b.astype(dtype), w.shifts, tol, w.max_iter)
    xs = {}
    for nslabs in (1, 2, 4, 8):
        S = make_slabs(ms, w, dtype, fmt, nslabs)
        g = ms.msolve_slabs_cgm(S, dev(w.b.astype(dtype)), w.shifts, tol, w.max_iter)
        xs[nslabs] = _check(w, dtype, tol, g, o)
        g2 = ms.msolve_slabs_cgm(S, dev(w.b.astype(dtype)), w.shifts, tol, w.max_iter)
        assert g2.iterations == g.iterations and torch.equal(g2.x, g.x)                # bit-reproducible
        assert ms.msolve_slabs_last_launch_count(S) > 0
        ms.msolve_slabs_destroy(S)
    for nslabs in (2, 4, 8):                                                           # across P: rounding only
        d = np.linalg.norm(xs[nslabs].astype(np.complex128) - xs[1]) / np.linalg.norm(xs[1])
        assert d <= (1e-11 if dtype == np.complex128 else 2e-5), (nslabs, d)


@pytest.mark.parametrize("fmt", ["csr", "bsr3"])
def test_slabs_bicgstabm_matches_oracle(ms, fmt):
    w = W.config3(extents=(8, 8, 8, 8))
    o = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, w.shifts, w.tol, w.max_iter)
    for nslabs in (2, 5):
        S = make_slabs(ms, w, np.complex128, fmt, nslabs)
        g = ms.msolve_slabs_bicgstabm(S, dev(w.b), w.shifts, w.tol, w.max_iter)
        _check(w, np.complex128, w.tol, g, o)
        ms.msolve_slabs_destroy(S)


def test_slabs_uneven_splits_real_and_edge_cases(ms):
    # real element type, hand-made splits (one slab much larger, one empty), the paper's matrix shape
    w = W.poisson_workload(40, 36, nshifts=6, real=True)
    splits = np.array([0, 400, 400, 1000, w.n], dtype=np.int64)
    S = ms.msolve_slabs_create_csr(w.rowptr, w.colidx, w.val, 4, splits=splits)
    g = ms.msolve_slabs_cgm(S, dev(w.b), w.shifts, 1e-10, w.max_iter)
    o = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 1e-10, w.max_iter)
    assert g.status == o.status == 0 and abs(g.iterations - o.iterations) <= 2
    x = g.x.cpu().numpy()
    for k in range(w.shifts.size):
        assert np.linalg.norm(x[k] - o.x[k]) <= 1e-9 * np.linalg.norm(o.x[k])
    # b = 0, max_iter = 0
    xb = torch.full((6, w.n), 7.0, dtype=torch.float64, device="cuda")
    r = ms.msolve_slabs_cgm(S, torch.zeros(w.n, dtype=torch.float64, device="cuda"), w.shifts, 1e-10, 50, x=xb)
    assert r.status == 0 and r.iterations == 0 and not r.x.abs().max().item()
    xb.fill_(7.0)
    r = ms.msolve_slabs_cgm(S, dev(w.b), w.shifts, 1e-10, 0, x=xb)
    assert r.status == ms.MSOLVE_MAXITER and not r.x.abs().max().item()
    ms.msolve_slabs_destroy(S)
    with pytest.raises(ms.MsolveError):                               # a split that is not 16-byte aligned in the vectors
        ms.msolve_slabs_create_csr(w.rowptr, w.colidx, w.val, 2, splits=np.array([0, 401, w.n], dtype=np.int64))
    with pytest.raises(ms.MsolveError):                               # splits that do not cover the rows / run backwards
        ms.msolve_slabs_create_csr(w.rowptr, w.colidx, w.val, 2, splits=np.array([0, 400, w.n + 4], dtype=np.int64))
    with pytest.raises(ms.MsolveError):
        ms.msolve_slabs_create_csr(w.rowptr, w.colidx, w.val, 3, splits=np.array([0, 800, 400, w.n], dtype=np.int64))
