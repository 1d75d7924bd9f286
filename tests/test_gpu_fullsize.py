"""Full-size parity in the launch configurations bench.py times (BASELINE configs[3] and [4]).

config 4 (32^3x64, N = 6.29 M, 16 shifts): the oracle runs the WHOLE solve on the host once per element type
(complex128 at tol 1e-10, complex64 at tol 1e-5, each on the same `.astype` inputs the GPU gets) and every
GPU variant -- BSR3, CSR (TMA-staged vector-CSR), merge-path CSR, the matrix-free lattice operator with each of
its three tile kernels, the TMA-staged fused update -- is compared with it element by element: per-shift
relative L2 difference, a max-abs bound on single elements, iteration counts, per-shift conv_iter, and true
residuals on sampled rows computed one by one in numpy.
config 5 (N = 2^22, 134 M nnz, 32 shifts): the same, whole solve, complex128 and complex64 (about 200 and 100
oracle iterations; the oracle is single-threaded, so this is the long test of the suite).
"""
import time

import numpy as np
import pytest
import torch

import oracle
from paper_1102_2143_b200 import workloads as W

pytestmark = pytest.mark.gpu

REL = {np.complex128: 1e-9, np.complex64: 1e-4}
MAXABS_C = 4.0


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


def compare_full(w, dtype, tol, res, ref, residual_shifts=None):
    """GPU SolveResult `res` against the oracle's MultishiftResult `ref`, every shift, element by element."""
    assert res.status == ref.status == 0
    assert abs(res.iterations - ref.iterations) <= 2, (res.iterations, ref.iterations)
    assert np.all(np.abs(res.conv_iter - ref.conv_iter) <= 2), (res.conv_iter, ref.conv_iter)
    rows = np.random.default_rng(0).integers(0, w.n, 2000)
    worst = 0.0
    for k, s in enumerate(w.shifts):
        xk = res.x[k].cpu().numpy()
        diff = xk.astype(np.complex128) - ref.x[k]
        d = np.linalg.norm(diff) / np.linalg.norm(ref.x[k])
        worst = max(worst, d)
        assert d <= REL[dtype], (k, d)
        assert np.abs(diff).max() <= MAXABS_C * REL[dtype] * np.abs(ref.x[k]).max(), (k, np.abs(diff).max())
        if residual_shifts is None or k in residual_shifts:
            rs = sampled_true_residual(w, xk.astype(np.complex128), s, rows)
            # ||b|| = 1: an rms residual entry of tol/sqrt(n) corresponds to ||r|| = tol
            assert np.sqrt(np.mean(np.abs(rs) ** 2) * w.n) <= 10 * tol, k
        assert res.relres[k] <= tol * (1 + 1e-12)
    return worst


# ------------------------------------------------------------------------------------------ config 4
@pytest.fixture(scope="module")
def c4():
    w = W.config4()
    refs = {}
    for dtype, tol in ((np.complex128, 1e-10), (np.complex64, 1e-5)):
        t0 = time.perf_counter()
        refs[dtype] = oracle.cgm(w.rowptr, w.colidx, w.val.astype(dtype), w.b.astype(dtype), w.shifts, tol, w.max_iter)
        print("oracle config 4 %s: %d iterations, %.1f s" % (np.dtype(dtype).name, refs[dtype].iterations, time.perf_counter() - t0))
    return w, refs


C4_VARIANTS = ["bsr3", "bsr3_stepwise", "bsr3_defer5", "csr", "csrmerge", "lat", "lat1", "lat2", "lat3", "lat4", "bsr3_updtma", "slabs8_bsr3", "slabs3_csr"]


def _c4_matrix(ms, w, dtype, variant):
    if variant == "slabs8_bsr3":        # row partition: 8 slabs along t (2 x 32^3 sites of halo per slab), csrc/slab.cu
        return ms.msolve_slabs_create_bsr3(w.browptr, w.bcolidx, w.blocks.astype(dtype), 8)
    if variant == "slabs3_csr":         # three slabs that do not divide the lattice evenly, TMA-staged vector-CSR per slab
        return ms.msolve_slabs_create_csr(w.rowptr, w.colidx, w.val.astype(dtype), 3)
    if variant in ("bsr3", "bsr3_updtma", "bsr3_stepwise", "bsr3_defer5"):
        A = ms.msolve_create_bsr3(dev(w.browptr), dev(w.bcolidx), dev(w.blocks.astype(dtype)))
        if variant == "bsr3_updtma":
            ms.msolve_config(A, ms.MSOLVE_CFG_UPDATE_KERNEL, 1)
        if variant == "bsr3_stepwise":   # x_k, p_k updated in every iteration (the default defers them, chunk of 32)
            ms.msolve_config(A, ms.MSOLVE_CFG_DEFER_UPDATE, 0)
        if variant == "bsr3_defer5":     # 24 (12) iterations = four full chunks and a partial one
            ms.msolve_config(A, ms.MSOLVE_CFG_DEFER_UPDATE, 5)
        return A
    if variant in ("csr", "csrmerge"):
        return ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val.astype(dtype)),
                                    ms.MSOLVE_SPMV_MERGE if variant == "csrmerge" else ms.MSOLVE_SPMV_AUTO)
    m = w.meta
    A = ms.msolve_create_lattice_su3(m["extents"], dev(w.links.astype(dtype)), m["diag"], m["c_f"], m["c_b"])
    if variant != "lat":
        ms.msolve_config(A, ms.MSOLVE_CFG_LATTICE_KERNEL, int(variant[3]))
    return A


@pytest.mark.parametrize("variant", C4_VARIANTS)
@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
def test_config4_full_vs_oracle(ms, c4, dtype, tol, variant):
    w, refs = c4
    A = _c4_matrix(ms, w, dtype, variant)
    if variant.startswith("slabs"):
        res = ms.msolve_slabs_cgm(A, dev(w.b.astype(dtype)), w.shifts, tol, w.max_iter)
        if variant == "slabs8_bsr3":     # every slab receives the two neighbouring time slices: 2 x 32^3 sites x 3 colours
            assert ms.msolve_slabs_halo_elements(A) == [2 * 32 * 32 * 32 * 3] * 8
    else:
        res = ms.msolve_cgm(A, dev(w.b.astype(dtype)), w.shifts, tol, w.max_iter)
    worst = compare_full(w, dtype, tol, res, refs[dtype], residual_shifts=(0, 7, 15))
    print("config 4 %s %s: %d iterations, worst relative L2 difference %.2e" % (np.dtype(dtype).name, variant, res.iterations, worst))
    (ms.msolve_slabs_destroy if variant.startswith("slabs") else ms.msolve_destroy)(A)
    del res, A
    torch.cuda.empty_cache()


def test_config4_full_multirhs_vs_oracle(ms, c4):
    # eq. (6) at the size bench.py times: three systems whose right-hand sides vary smoothly with the shift
    w, _ = c4
    shifts = np.array([0.0, 0.3, 1.0])
    rng = np.random.default_rng(51)
    c = rng.standard_normal((2, w.n)) + 1j * rng.standard_normal((2, w.n))
    g = rng.standard_normal((3, w.n)) + 1j * rng.standard_normal((3, w.n))
    B = np.array([c[0] + t * c[1] + 0.05 * g[i] for i, t in enumerate(shifts)])
    B /= np.linalg.norm(B[0])
    del c, g
    A = ms.msolve_create_bsr3(dev(w.browptr), dev(w.bcolidx), dev(w.blocks))
    res = ms.msolve_solve_multirhs(A, ms.MSOLVE_ALG_CGM, dev(B), shifts, 1e-10, w.max_iter)
    ref = oracle.multirhs(w.rowptr, w.colidx, w.val, B, shifts, 1e-10, w.max_iter)
    assert res.status == ref.status == 0 and abs(res.iterations - ref.iterations) <= 2
    rows = np.random.default_rng(0).integers(0, w.n, 2000)
    for k, s in enumerate(shifts):
        xk = res.x[k].cpu().numpy()
        diff = xk - ref.x[k]
        assert np.linalg.norm(diff) <= 1e-9 * np.linalg.norm(ref.x[k]), k
        assert np.abs(diff).max() <= MAXABS_C * 1e-9 * np.abs(ref.x[k]).max(), k
        out = np.empty(rows.size, dtype=np.complex128)
        for t, i in enumerate(rows):
            lo, hi = w.rowptr[i], w.rowptr[i + 1]
            out[t] = B[k, i] - (np.dot(w.val[lo:hi], xk[w.colidx[lo:hi]]) + s * xk[i])
        assert np.sqrt(np.mean(np.abs(out) ** 2) * w.n) <= 10 * 1e-10 * np.linalg.norm(B[k]), k
    ms.msolve_destroy(A)


# ------------------------------------------------------------------------------------------ config 5
@pytest.fixture(scope="module")
def c5():
    return W.config5()


@pytest.mark.parametrize("dtype,tol", [(np.complex64, 1e-5), (np.complex128, 1e-10)])
def test_config5_full_vs_oracle(ms, c5, dtype, tol):
    w = c5
    val, b = w.val.astype(dtype), w.b.astype(dtype)
    A = ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(val))
    res = ms.msolve_cgm(A, dev(b), w.shifts, tol, w.max_iter)
    assert res.status == 0
    assert np.all(np.diff(res.conv_iter) <= 0) and res.iterations == res.conv_iter.max()
    t0 = time.perf_counter()
    ref = oracle.cgm(w.rowptr, w.colidx, val, b, w.shifts, tol, w.max_iter)
    print("oracle config 5 %s: %d iterations, %.1f s" % (np.dtype(dtype).name, ref.iterations, time.perf_counter() - t0))
    worst = compare_full(w, dtype, tol, res, ref, residual_shifts=(0, 13, 31))
    print("config 5 %s: %d iterations, worst relative L2 difference %.2e" % (np.dtype(dtype).name, res.iterations, worst))
    ms.msolve_destroy(A)
    del res, A
    torch.cuda.empty_cache()
    if dtype == np.complex128:
        # the merge-path kernel on the same matrix against the same oracle result
        A = ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(val), ms.MSOLVE_SPMV_MERGE)
        res = ms.msolve_cgm(A, dev(b), w.shifts, tol, w.max_iter)
        compare_full(w, dtype, tol, res, ref, residual_shifts=())
        ms.msolve_destroy(A)
