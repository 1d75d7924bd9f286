"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Bars are BASELINE.json's: per-shift relative L2 difference <= 1e-9
(complex128) / 1e-4 (complex64), true residual <= 10 tol, iteration counts within +-2.
Run with `pytest -m gpu` on the B200 box."""
import numpy as np
import pytest
import scipy.sparse as sp
import torch

import oracle
from paper_1102_2143_b200 import workloads as W

pytestmark = pytest.mark.gpu

REL = {np.complex128: 1e-9, np.complex64: 1e-4}
TORCH = {np.complex128: torch.complex128, np.complex64: torch.complex64}
MAXABS_C = 4.0


@pytest.fixture(scope="module")
def ms():
    from paper_1102_2143_b200 import binding, build
    build.build()
    binding.load_library()
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


FORCED_CFG = {}     # msolve_config options applied to every handle make_matrix creates (set by fixtures)


def make_matrix(ms, w, dtype, fmt, flags=0, cfg=None):
    A = _create(ms, w, dtype, fmt, flags)
    # The tests of this file exercise the iteration as a graph of kernels at every size (by default the library
    # would run systems this small as one cooperative kernel: tests/test_gpu_fused.py covers that path).
    base = {ms.MSOLVE_CFG_ITER_PATH: 1}
    for key, value in list(base.items()) + list(FORCED_CFG.items()) + list((cfg or {}).items()):
        ms.msolve_config(A, key, value)
    return A


def _create(ms, w, dtype, fmt, flags):
    if fmt == "bsr3rows":   # the simple one-thread-per-row BSR3 kernel instead of the TMA-staged one
        return ms.msolve_create_bsr3(dev(w.browptr), dev(w.bcolidx), dev(w.blocks.astype(dtype)), ms.MSOLVE_SPMV_VECTOR)
    if fmt in ("lat", "latrows"):   # matrix-free operator from the link field (TMA tile kernel / row kernel)
        m = w.meta
        return ms.msolve_create_lattice_su3(m["extents"], dev(w.links.astype(dtype)), m["diag"], m["c_f"], m["c_b"],
                                            ms.MSOLVE_SPMV_VECTOR if fmt == "latrows" else ms.MSOLVE_SPMV_AUTO)
    if fmt == "bsr3":
        return ms.msolve_create_bsr3(dev(w.browptr), dev(w.bcolidx), dev(w.blocks.astype(dtype)))
    if fmt == "csrmerge":   # merge-path CSR forced (AUTO picks it only for irregular rows)
        return ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val.astype(dtype)), ms.MSOLVE_SPMV_MERGE)
    if fmt == "csrtile":    # TMA-staged vector-CSR forced (AUTO picks it for large matrices of short rows)
        return ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val.astype(dtype)), ms.MSOLVE_SPMV_TILE)
    if fmt == "csrvector":
        return ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val.astype(dtype)), ms.MSOLVE_SPMV_VECTOR)
    return ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val.astype(dtype)), flags)


def gpu_solve(ms, w, dtype, fmt, tol=None, max_iter=None, shifts=None, flags=0, cfg=None):
    A = make_matrix(ms, w, dtype, fmt, flags, cfg)
    fn = ms.msolve_cgm if w.algorithm == "cgm" else ms.msolve_bicgstabm
    res = fn(A, dev(w.b.astype(dtype)), w.shifts if shifts is None else shifts,
             w.tol if tol is None else tol, w.max_iter if max_iter is None else max_iter)
    torch.cuda.synchronize()
    out = (res.status, res.iterations, res.x.cpu().numpy(), res.conv_iter.copy(), res.relres.copy())
    launches = ms.msolve_last_launch_count(A)
    ms.msolve_destroy(A)
    return out + (launches,)


def oracle_solve(w, dtype, tol=None, max_iter=None, shifts=None):
    fn = oracle.cgm if w.algorithm == "cgm" else oracle.bicgstabm
    return fn(w.rowptr, w.colidx, w.val.astype(dtype), w.b.astype(dtype), w.shifts if shifts is None else shifts,
              w.tol if tol is None else tol, w.max_iter if max_iter is None else max_iter)


def check_parity(w, dtype, g, o, tol):
    status, it, x, conv, rel, _ = g
    assert status == o.status == oracle.OK
    assert abs(it - o.iterations) <= 2
    assert np.all(np.abs(conv - o.conv_iter) <= 2)
    A = sp.csr_matrix((w.val, w.colidx, w.rowptr), shape=(w.n, w.n))
    for k, s in enumerate(w.shifts):
        diff = x[k].astype(np.complex128) - o.x[k].astype(np.complex128)
        d = np.linalg.norm(diff) / np.linalg.norm(o.x[k])
        assert d <= REL[dtype], (k, d)
        # element by element: no single entry may be off by more than MAXABS_C bars of the largest entry (a norm
        # alone lets one wrong element in millions through at the complex64 bar)
        assert np.abs(diff).max() <= MAXABS_C * REL[dtype] * np.abs(o.x[k]).max(), (k, np.abs(diff).max())
        xk = x[k].astype(np.complex128)
        true = np.linalg.norm(w.b - (A @ xk + s * xk)) / np.linalg.norm(w.b)
        assert true <= 10.0 * tol, (k, true)
        assert rel[k] <= tol * (1 + 1e-12)


# ------------------------------------------------------------------------------- SpMV
@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("which,fmt", [("c1", "csr"), ("c2", "csr"), ("c2", "bsr3"), ("c2", "bsr3rows"),
                                       ("c2big", "bsr3"), ("c5", "csr"), ("c5", "csrvector"), ("c5", "csrmerge"),
                                       ("c1", "csrmerge"), ("c2big", "csrmerge"), ("c5big", "csrmerge"),
                                       ("c1", "csrtile"), ("c2", "csrtile"), ("c2big", "csrtile")])
def test_spmv_matches_oracle(ms, dtype, which, fmt):
    w = {"c1": lambda: W.config1(), "c2": lambda: W.config2(extents=(4, 4, 6, 5)),
         "c2big": lambda: W.config2(extents=(12, 10, 9, 11)),   # 11880 sites: many tiles per CTA, ragged tail
         "c5": lambda: W.config5(n=5003), "c5big": lambda: W.config5(n=200003)}[which]()
    rng = np.random.default_rng(3)
    x = (rng.standard_normal(w.n) + 1j * rng.standard_normal(w.n)).astype(dtype)
    A = make_matrix(ms, w, dtype, fmt)
    y, dot = ms.msolve_spmv(A, dev(x))
    y = y.cpu().numpy()
    ref = oracle.spmv(w.rowptr, w.colidx, w.val.astype(dtype), x)
    eps = 1e-13 if dtype == np.complex128 else 1e-5
    assert np.linalg.norm(y - ref) / np.linalg.norm(ref) < eps
    ref_dot = np.vdot(x.astype(np.complex128), ref.astype(np.complex128))
    assert abs(dot - ref_dot) / abs(ref_dot) < eps
    ms.msolve_destroy(A)


def _random_csr(rng, lengths, n):
    rowptr = np.zeros(n + 1, dtype=np.int32)
    rowptr[1:] = np.cumsum(lengths)
    nnz = int(rowptr[-1])
    colidx = rng.integers(0, n, nnz).astype(np.int32)
    val = (rng.standard_normal(nnz) + 1j * rng.standard_normal(nnz))
    return rowptr, colidx, val


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("shape", ["empty_rows", "one_long_row", "long_rows_mixed", "all_empty", "single_row", "tiny"])
def test_merge_path_degenerate_rows(ms, dtype, shape):
    # merge-path tiles cut rows anywhere: empty rows (also in floods at a tile boundary), rows
    # spanning many tiles, matrices smaller than one tile.  Not a solver workload: SpMV only.
    rng = np.random.default_rng(11)
    if shape == "empty_rows":
        n = 30011
        lengths = rng.integers(0, 40, n) * (rng.random(n) < 0.3)
        lengths[5000:12000] = 0                                   # a flood of empty rows
    elif shape == "one_long_row":
        n = 4099
        lengths = np.full(n, 3)
        lengths[1234] = 50001                                     # spans ~25-50 tiles
    elif shape == "long_rows_mixed":
        n = 2500
        lengths = rng.integers(1, 12, n)
        lengths[rng.integers(0, n, 12)] = rng.integers(1500, 9000, 12)
        lengths[-1] = 4097                                        # long last row
        lengths[0] = 3000                                         # long first row
    elif shape == "all_empty":
        n = 5000
        lengths = np.zeros(n, dtype=np.int64)
    elif shape == "single_row":
        n = 1
        lengths = np.array([1])
    else:
        n = 7
        lengths = np.array([0, 2, 0, 0, 5, 1, 0])
    rowptr, colidx, val = _random_csr(rng, lengths, n)
    if colidx.size == 0:                                          # keep the arrays non-NULL
        colidx_d, val_d = torch.zeros(4, dtype=torch.int32, device="cuda"), torch.zeros(4, dtype=TORCH[dtype], device="cuda")
        A = ms.msolve_create_csr(dev(rowptr), colidx_d[:0], val_d[:0], ms.MSOLVE_SPMV_MERGE)
    else:
        A = ms.msolve_create_csr(dev(rowptr), dev(colidx), dev(val.astype(dtype)), ms.MSOLVE_SPMV_MERGE)
    x = (rng.standard_normal(n) + 1j * rng.standard_normal(n)).astype(dtype)
    y, dot = ms.msolve_spmv(A, dev(x), torch.full((n,), 7.0, dtype=TORCH[dtype], device="cuda"))
    y = y.cpu().numpy()
    ref = oracle.spmv(rowptr, colidx, val.astype(dtype), x)
    eps = 1e-13 if dtype == np.complex128 else 2e-5
    scale = max(np.linalg.norm(ref), 1e-300)
    assert np.linalg.norm(y - ref) <= eps * scale
    assert np.array_equal(y[lengths == 0], np.zeros(int((lengths == 0).sum()), dtype=dtype))   # every row written
    ref_dot = np.vdot(x.astype(np.complex128), ref.astype(np.complex128))
    assert abs(dot - ref_dot) <= eps * max(abs(ref_dot), np.linalg.norm(x) * scale)
    # bit-reproducible: a second launch gives the same bytes
    y2, dot2 = ms.msolve_spmv(A, dev(x))
    assert np.array_equal(y2.cpu().numpy(), y) and dot2 == dot
    ms.msolve_destroy(A)


# ------------------------------------------------------------------------------- CG-M
def test_config1_cgm_c128(ms):
    w = W.config1()
    g = gpu_solve(ms, w, np.complex128, "csr")
    o = oracle_solve(w, np.complex128)
    check_parity(w, np.complex128, g, o, w.tol)
    assert g[5] == 2 + 6 * g[1]          # init + 6 kernels per iteration (the sixth is the deferred update's flush), no host round trips


@pytest.mark.parametrize("fmt", ["csr", "bsr3", "bsr3rows"])
@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
def test_config2_cgm(ms, fmt, dtype, tol):
    w = W.config2()
    g = gpu_solve(ms, w, dtype, fmt, tol=tol)
    o = oracle_solve(w, dtype, tol=tol)
    check_parity(w, dtype, g, o, tol)


@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
@pytest.mark.parametrize("extents", [(8, 8, 8, 8), (6, 5, 7, 9)])     # 1890 sites: tiles with a ragged tail
def test_update_kernels_agree(ms, extents, dtype, tol):
    # the register kernel (default) and the TMA-staged fused update do the same arithmetic
    w = W.config2(extents=extents)
    o = oracle_solve(w, dtype, tol=tol)
    xs = []
    for which in (0, 1):
        g = gpu_solve(ms, w, dtype, "bsr3", tol=tol, cfg={ms.MSOLVE_CFG_UPDATE_KERNEL: which})
        check_parity(w, dtype, g, o, tol)
        xs.append(g[2])
    d = np.linalg.norm(xs[0].astype(np.complex128) - xs[1]) / np.linalg.norm(xs[1])
    assert d <= (1e-12 if dtype == np.complex128 else 1e-5)


@pytest.mark.parametrize("fmt", ["csr", "csrtile", "bsr3"])
@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
def test_config4_scaled_cgm(ms, fmt, dtype, tol):
    w = W.config4(extents=(8, 8, 8, 16), tol=tol)
    g = gpu_solve(ms, w, dtype, fmt)
    o = oracle_solve(w, dtype)
    check_parity(w, dtype, g, o, tol)


@pytest.mark.parametrize("fmt", ["csr", "csrvector", "csrmerge"])
@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
def test_config5_scaled_cgm(ms, fmt, dtype, tol):
    w = W.config5(n=(1 << 15) + 37, tol=tol)       # ragged size; "csr" = AUTO (vector kernel: rows <= 200)
    g = gpu_solve(ms, w, dtype, fmt)
    o = oracle_solve(w, dtype)
    check_parity(w, dtype, g, o, tol)
    assert np.all(np.diff(g[3]) <= 0)              # larger shifts never converge later
    per_iter = 7 if fmt == "csrmerge" else 6       # 6 kernels (the sixth: the deferred update's flush); merge-path SpMV = tile kernel + carry fix-up
    assert g[5] == 2 + per_iter * g[1]


def test_bicgstabm_csr_tile(ms):
    # both SpMV roles of BiCGStab-M through the TMA-staged vector-CSR kernel
    w = W.config3(extents=(6, 6, 6, 6))
    g = gpu_solve(ms, w, np.complex128, "csrtile")
    o = oracle_solve(w, np.complex128)
    check_parity(w, np.complex128, g, o, w.tol)
    assert g[5] == 2 + 7 * g[1]


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("shape", ["ragged", "empty_rows", "max_rows", "all_empty", "single_row", "tiny", "short", "mid", "long_f"])
def test_csr_tile_degenerate_rows(ms, dtype, shape):
    # TMA-staged vector-CSR: rows of 0..64 non-zeros in any mix (lane counts 2..16), tiles whose
    # non-zero range starts and ends off the 4-element alignment, matrices smaller than one tile
    rng = np.random.default_rng(17)
    if shape == "ragged":
        n, lengths = 30011, rng.integers(0, 28, 30011)
    elif shape == "empty_rows":
        n = 20001
        lengths = rng.integers(1, 16, n) * (rng.random(n) < 0.4)
        lengths[3000:9000] = 0
    elif shape == "max_rows":
        n, lengths = 5003, rng.integers(40, 65, 5003)
    elif shape == "all_empty":
        n, lengths = 5000, np.zeros(5000, dtype=np.int64)
    elif shape == "single_row":
        n, lengths = 1, np.array([1])
    elif shape == "tiny":
        n, lengths = 7, np.array([0, 2, 0, 0, 5, 1, 0])
    elif shape == "mid":
        n, lengths = 9001, rng.integers(9, 17, 9001)              # 4 lanes x 4
    elif shape == "long_f":
        n, lengths = 3001, rng.integers(90, 129, 3001)            # 16 lanes x 8: elements of <= 8 bytes only
    else:
        n, lengths = 40007, rng.integers(1, 6, 40007)
    rowptr, colidx, val = _random_csr(rng, lengths, n)
    if shape == "long_f" and dtype == np.complex128:
        with pytest.raises(Exception):                            # 16-byte elements: rows of at most 64
            ms.msolve_create_csr(dev(rowptr), dev(colidx), dev(val.astype(dtype)), ms.MSOLVE_SPMV_TILE)
        return
    if colidx.size == 0:
        colidx_d, val_d = torch.zeros(4, dtype=torch.int32, device="cuda"), torch.zeros(4, dtype=TORCH[dtype], device="cuda")
        with pytest.raises(Exception):                            # no non-zeros: not a tile-kernel matrix
            ms.msolve_create_csr(dev(rowptr), colidx_d[:0], val_d[:0], ms.MSOLVE_SPMV_TILE)
        return
    A = ms.msolve_create_csr(dev(rowptr), dev(colidx), dev(val.astype(dtype)), ms.MSOLVE_SPMV_TILE)
    x = (rng.standard_normal(n) + 1j * rng.standard_normal(n)).astype(dtype)
    y, dot = ms.msolve_spmv(A, dev(x), torch.full((n,), 7.0, dtype=TORCH[dtype], device="cuda"))
    y = y.cpu().numpy()
    ref = oracle.spmv(rowptr, colidx, val.astype(dtype), x)
    eps = 1e-13 if dtype == np.complex128 else 2e-5
    scale = max(np.linalg.norm(ref), 1e-300)
    assert np.linalg.norm(y - ref) <= eps * scale
    assert np.array_equal(y[lengths == 0], np.zeros(int((lengths == 0).sum()), dtype=dtype))   # every row written
    ref_dot = np.vdot(x.astype(np.complex128), ref.astype(np.complex128))
    assert abs(dot - ref_dot) <= eps * max(abs(ref_dot), np.linalg.norm(x) * scale)
    y2, dot2 = ms.msolve_spmv(A, dev(x))
    assert np.array_equal(y2.cpu().numpy(), y) and dot2 == dot
    ms.msolve_destroy(A)


def test_csr_tile_rejects_long_rows(ms):
    rng = np.random.default_rng(5)
    lengths = np.full(100, 4)
    lengths[17] = 65
    rowptr, colidx, val = _random_csr(rng, lengths, 100)
    with pytest.raises(Exception):
        ms.msolve_create_csr(dev(rowptr), dev(colidx), dev(val), ms.MSOLVE_SPMV_TILE)


def test_bicgstabm_merge_path(ms):
    # both SpMV roles of BiCGStab-M (incl. the quadratic <t,t> on rows cut by tile boundaries)
    w = W.config3(extents=(6, 6, 6, 6))
    g = gpu_solve(ms, w, np.complex128, "csrmerge")
    o = oracle_solve(w, np.complex128)
    check_parity(w, np.complex128, g, o, w.tol)
    assert g[5] == 2 + 9 * g[1]


# ------------------------------------------------------------------------------- BiCGStab-M
@pytest.mark.parametrize("fmt", ["csr", "bsr3"])
def test_config3_bicgstabm_c128(ms, fmt):
    w = W.config3()                                 # full size: 16^4, N = 196608
    g = gpu_solve(ms, w, np.complex128, fmt)
    o = oracle_solve(w, np.complex128)
    check_parity(w, np.complex128, g, o, w.tol)
    assert g[5] == 2 + 7 * g[1]


def test_config3_scaled_bicgstabm_c64(ms):
    w = W.config3(extents=(8, 8, 8, 8))
    g = gpu_solve(ms, w, np.complex64, "bsr3", tol=1e-5)
    o = oracle_solve(w, np.complex64, tol=1e-5)
    check_parity(w, np.complex64, g, o, 1e-5)


# ------------------------------------------------------------------------------- edge cases
def test_zero_rhs_and_zero_iterations(ms):
    w = W.config1()
    A = make_matrix(ms, w, np.complex128, "csr")
    x = torch.full((4, w.n), 7.0, dtype=torch.complex128, device="cuda")
    res = ms.msolve_cgm(A, torch.zeros(w.n, dtype=torch.complex128, device="cuda"), w.shifts, 1e-10, 100, x=x)
    assert res.status == ms.MSOLVE_OK and res.iterations == 0 and not res.x.abs().max().item()
    assert np.all(res.conv_iter == 0)
    x.fill_(7.0)
    res = ms.msolve_cgm(A, dev(w.b), w.shifts, 1e-10, 0, x=x)
    assert res.status == ms.MSOLVE_MAXITER and res.iterations == 0 and not res.x.abs().max().item()
    ms.msolve_destroy(A)


@pytest.mark.parametrize("alg", ["cgm", "bicgstabm"])
def test_maxiter_matches_oracle_iterate(ms, alg):
    # stopped early, the GPU iterate equals the oracle's iterate at the same n
    w = W.config2(extents=(4, 4, 4, 4)) if alg == "cgm" else W.config3(extents=(4, 4, 4, 4))
    for nit in (1, 2, 5):
        g = gpu_solve(ms, w, np.complex128, "csr", tol=0.0, max_iter=nit)
        o = oracle_solve(w, np.complex128, tol=0.0, max_iter=nit)
        assert g[0] == o.status == oracle.MAXITER and g[1] == o.iterations == nit
        for k in range(w.shifts.size):
            assert np.linalg.norm(g[2][k] - o.x[k]) / np.linalg.norm(o.x[k]) < 1e-12
        assert np.allclose(g[4], o.relres, rtol=1e-10)


def test_odd_length_c64_and_duplicate_shifts(ms):
    w = W.config5(n=2051, tol=1e-5)                # odd n: 8-byte access path for complex64
    shifts = np.array([0.5, 0.5, 0.001, 3.0])      # unsorted, duplicated
    g = gpu_solve(ms, w, np.complex64, "csr", shifts=shifts)
    o = oracle_solve(w, np.complex64, shifts=shifts)
    w.shifts = shifts
    check_parity(w, np.complex64, g, o, 1e-5)
    assert np.array_equal(g[2][0], g[2][1])


def test_max_shifts_and_too_many(ms):
    w = W.config1()
    shifts = np.linspace(0.0, 2.0, ms.MSOLVE_MAX_SHIFTS)
    g = gpu_solve(ms, w, np.complex128, "csr", shifts=shifts)
    o = oracle_solve(w, np.complex128, shifts=shifts)
    w.shifts = shifts
    check_parity(w, np.complex128, g, o, w.tol)
    A = make_matrix(ms, w, np.complex128, "csr")
    with pytest.raises(ms.MsolveError):
        ms.msolve_cgm(A, dev(w.b), np.zeros(ms.MSOLVE_MAX_SHIFTS + 1), 1e-10, 10)
    ms.msolve_destroy(A)


@pytest.mark.parametrize("path", [1, 2], ids=["graph", "fused"])
def test_breakdown_reported(ms, path):
    # indefinite A: <p,Ap> < 0 in the first loop body (R16).  The iterate at that point is x_k = 0, which is what
    # the oracle returns; d_x must be fully overwritten with it (include/msolve.h), not left as the caller had it.
    n = 64
    rowptr = np.arange(n + 1, dtype=np.int32)
    colidx = np.arange(n, dtype=np.int32)
    val = -np.ones(n, dtype=np.complex128)
    b = W.unit_rhs(1, n)
    A = ms.msolve_create_csr(dev(rowptr), dev(colidx), dev(val))
    ms.msolve_config(A, ms.MSOLVE_CFG_ITER_PATH, path)
    x = torch.full((2, n), 7.0, dtype=torch.complex128, device="cuda")
    res = ms.msolve_cgm(A, dev(b), [0.0, 0.5], 1e-10, 10, x=x)
    o = oracle.cgm(rowptr, colidx, val, b, [0.0, 0.5], 1e-10, 10)
    assert res.status == ms.MSOLVE_BREAKDOWN == o.status and res.iterations == o.iterations == 0
    assert np.array_equal(res.x.cpu().numpy(), o.x) and not o.x.any()
    ms.msolve_destroy(A)
    # BiCGStab-M, <r0, A p> = 0 exactly in the first loop body (A swaps neighbouring entries, b lives on the even
    # ones): breakdown before any update, x = 0
    rp2 = np.arange(n + 1, dtype=np.int32)
    ci2 = (np.arange(n) ^ 1).astype(np.int32)
    v2 = np.ones(n, dtype=np.complex128)
    b2 = np.zeros(n, dtype=np.complex128)
    b2[::2] = W.unit_rhs(2, n // 2)
    A = ms.msolve_create_csr(dev(rp2), dev(ci2), dev(v2))
    ms.msolve_config(A, ms.MSOLVE_CFG_ITER_PATH, path)
    x.fill_(7.0)
    res = ms.msolve_bicgstabm(A, dev(b2), [0.0, 0.5], 1e-10, 10, x=x)
    o = oracle.bicgstabm(rp2, ci2, v2, b2, [0.0, 0.5], 1e-10, 10)
    assert res.status == ms.MSOLVE_BREAKDOWN == o.status and res.iterations == o.iterations == 0
    assert np.array_equal(res.x.cpu().numpy(), o.x) and not o.x.any()
    ms.msolve_destroy(A)
    # BiCGStab-M on A = c I (R17): s = r + beta q vanishes after the first half step up to rounding.  Whether that is
    # an exact zero (<t,t> = 0: breakdown, x = 0, what the oracle's unfused arithmetic gives) or a residual of one
    # ulp (one more half step on rounding noise: converged, x_k = b / (c + sigma_k)) is decided by the rounding of
    # one multiply-add; both are correct outcomes and nothing else is.
    c = 2.5
    val = np.full(n, c, dtype=np.complex128)
    A = ms.msolve_create_csr(dev(rowptr), dev(colidx), dev(val))
    ms.msolve_config(A, ms.MSOLVE_CFG_ITER_PATH, path)
    x.fill_(7.0)
    res = ms.msolve_bicgstabm(A, dev(b), [0.0, 0.5], 1e-10, 10, x=x)
    xg = res.x.cpu().numpy()
    if res.status == ms.MSOLVE_BREAKDOWN:
        assert res.iterations == 0 and not xg.any()
    else:
        assert res.status == ms.MSOLVE_OK and res.iterations == 1
        for k, sg in enumerate([0.0, 0.5]):
            assert np.linalg.norm(xg[k] - b / (c + sg)) <= 1e-14 * np.linalg.norm(b)
    ms.msolve_destroy(A)
    # a breakdown AFTER the first update keeps the iterate reached so far (same as the oracle)
    val = np.ones(n, dtype=np.complex128)
    val[n // 2:] = -1.0                                   # indefinite, but <b,Ab> > 0 for this b
    bb = np.zeros(n, dtype=np.complex128)
    bb[: n // 2] = 1.0
    bb[n // 2:] = 0.5
    bb /= np.linalg.norm(bb)
    A = ms.msolve_create_csr(dev(rowptr), dev(colidx), dev(val))
    ms.msolve_config(A, ms.MSOLVE_CFG_ITER_PATH, path)
    res = ms.msolve_cgm(A, dev(bb), [0.0], 1e-10, 10)
    o = oracle.cgm(rowptr, colidx, val, bb, [0.0], 1e-10, 10)
    assert res.status == o.status and res.iterations == o.iterations
    if o.status == oracle.BREAKDOWN and o.iterations > 0:
        assert np.linalg.norm(res.x.cpu().numpy() - o.x) <= 1e-12 * np.linalg.norm(o.x)
    ms.msolve_destroy(A)


# ------------------------------------------------------------------------------- stop rule, scalar history
@pytest.mark.parametrize("alg", ["cgm", "bicgstabm"])
@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
def test_stop_rule_base_matches_oracle(ms, alg, dtype, tol):
    # MSOLVE_CFG_STOP_RULE = 1: Alg. 1 l.15 read literally: iterate until the UNSHIFTED residual is
    # below tol, no shift is frozen before that.  Shifts without sigma = 0, so the two rules really differ.
    w = W.config2(extents=(4, 6, 4, 6)) if alg == "cgm" else W.config3(extents=(4, 6, 4, 6))
    shifts = np.array([0.7, 0.01, 0.15, 3.0])
    g = gpu_solve(ms, w, dtype, "bsr3", tol=tol, shifts=shifts, cfg={ms.MSOLVE_CFG_STOP_RULE: 1})
    ofn = oracle.cgm if alg == "cgm" else oracle.bicgstabm
    o = ofn(w.rowptr, w.colidx, w.val.astype(dtype), w.b.astype(dtype), shifts, tol, w.max_iter, stop_rule=1)
    o0 = ofn(w.rowptr, w.colidx, w.val.astype(dtype), w.b.astype(dtype), shifts, tol, w.max_iter, stop_rule=0)
    assert o.iterations > o0.conv_iter.min()                    # the literal rule runs longer than the fastest shift
    assert g[0] == o.status == oracle.OK and abs(g[1] - o.iterations) <= 2
    assert np.all(g[3] == g[1]) and np.all(o.conv_iter == o.iterations)
    for k in range(shifts.size):
        diff = g[2][k].astype(np.complex128) - o.x[k]
        assert np.linalg.norm(diff) <= REL[dtype] * np.linalg.norm(o.x[k]), k
        assert np.abs(diff).max() <= MAXABS_C * REL[dtype] * np.abs(o.x[k]).max(), k
    if g[1] == o.iterations:
        assert np.allclose(g[4], o.relres, rtol=1e-6 if dtype == np.complex128 else 1e-2)


HIST_RTOL = 1e-12
HIST_ULPS = 64.0


@pytest.mark.parametrize("which,fmt", [("c1", "csr"), ("c2", "bsr3"), ("c2", "csr"), ("c3", "bsr3"), ("c3", "csr")])
def test_scalar_history_matches_oracle(ms, which, fmt):
    # SURVEY 8(c) C6 "brute force": the scalars of Alg. 1 l.20-26 that the scalar kernels
    # produce -- beta, alpha, R1 and zeta / beta_k / alpha_k (chi_k) of every shift, every iteration -- against
    # the oracle's record of the same quantities, on configs 1, 2 and the 4^4 config 3.
    w = {"c1": W.config1, "c2": W.config2, "c3": lambda: W.config3(extents=(4, 4, 4, 4))}[which]()
    S = w.shifts.size
    cols = 3 + 3 * S if w.algorithm == "cgm" else 8 + 6 * S
    cap = 64
    A = make_matrix(ms, w, np.complex128, fmt)
    hist = torch.zeros((cap, cols), dtype=torch.float64, device="cuda")
    ms.msolve_set_history(A, hist)
    fn, ofn = (ms.msolve_cgm, oracle.cgm) if w.algorithm == "cgm" else (ms.msolve_bicgstabm, oracle.bicgstabm)
    res = fn(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    o = ofn(w.rowptr, w.colidx, w.val, w.b, w.shifts, w.tol, w.max_iter, hist_cap=cap)
    assert res.status == o.status == 0 and res.iterations == o.iterations <= cap
    hg = hist.cpu().numpy()[: o.iterations]
    assert not hist.cpu().numpy()[o.iterations:].any()              # nothing written past the last iteration
    if w.algorithm == "cgm":
        dev_rel = np.abs(hg - o.hist) / np.abs(o.hist)
        rr = o.hist[:, 2]
    else:                                                           # complex pairs: relative to the modulus
        zg = np.concatenate([hg[:, :6].copy().view(np.complex128), hg[:, 8:].copy().view(np.complex128)], axis=1)
        zo = np.concatenate([o.hist[:, :6].copy().view(np.complex128), o.hist[:, 8:].copy().view(np.complex128)], axis=1)
        rr = o.hist[:, 6]
        dev_rel = np.concatenate([np.abs(zg - zo) / np.abs(zo), (np.abs(hg[:, 6] - rr) / rr)[:, None]], axis=1)
        assert not hg[:, 7].any()
    # The bar: both sides run the same recurrences; they differ in the summation order of the
    # dots and in fused multiply-adds, i.e. by a few ulp of ||b|| per element of r and per iteration.  Relative to
    # the shrinking residual that is (n + 1) eps ||b|| / ||r_n||, so a scalar of iteration n may deviate by
    # HIST_RTOL + HIST_ULPS (n + 1) eps ||b|| / ||r_{n+1}|| -- 1e-12 while the residual is large, where a wrong
    # formula shows as an O(1) deviation.
    bar = HIST_RTOL + HIST_ULPS * np.finfo(np.float64).eps * (np.arange(o.iterations) + 1) / np.sqrt(rr)
    print("history %s/%s: max relative deviation per iteration" % (which, fmt), dev_rel.max(axis=1), "bar", bar)
    assert np.all(dev_rel.max(axis=1) <= bar), (dev_rel.max(axis=1) / bar).max()
    # switching it off: the next solve leaves the buffer alone
    ms.msolve_set_history(A, None)
    hist.zero_()
    fn(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    assert not hist.any().item()
    # a short buffer: rows beyond cap are dropped, the rest is the same
    short = torch.zeros((3, cols), dtype=torch.float64, device="cuda")
    ms.msolve_set_history(A, short)
    fn(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    assert np.array_equal(short.cpu().numpy(), hg[:3])
    ms.msolve_destroy(A)


def test_chunked_loop_mode_same_result(ms):
    w = W.config2(extents=(4, 4, 4, 4))
    a = gpu_solve(ms, w, np.complex128, "bsr3")
    b = gpu_solve(ms, w, np.complex128, "bsr3", cfg={ms.MSOLVE_CFG_LOOP_MODE: 1})
    assert a[1] == b[1] and np.array_equal(a[2], b[2]) and np.array_equal(a[3], b[3])


def test_handle_reuse_and_solve_host(ms):
    w = W.config2(extents=(4, 4, 4, 4))
    A = make_matrix(ms, w, np.complex128, "bsr3")
    r1 = ms.msolve_cgm(A, dev(w.b), w.shifts, w.tol, 500)
    r2 = ms.msolve_cgm(A, dev(w.b), w.shifts[:3], w.tol, 500)        # other S, same cached graph
    assert torch.equal(r1.x[:3], r2.x) and np.array_equal(r1.conv_iter[:3], r2.conv_iter)
    rh = ms.msolve_solve_host(A, ms.MSOLVE_ALG_CGM, torch.from_numpy(w.b), w.shifts, w.tol, 500)
    assert not rh.x.is_cuda and torch.equal(rh.x, r1.x.cpu()) and rh.iterations == r1.iterations
    ms.msolve_destroy(A)


@pytest.mark.parametrize("alg", ["cgm", "bicgstabm"])
def test_solve_host_batch_matches_single_solves(ms, alg):
    # five right-hand sides through the pipelined batch call (two device slots in turn, D2H of solve i
    # overlapping solve i+1): every solution set equals the one of a single host call, bit for bit
    w = W.config2(extents=(8, 6, 4, 6)) if alg == "cgm" else W.config3(extents=(6, 6, 4, 6))
    A = make_matrix(ms, w, np.complex128, "bsr3")
    code = ms.MSOLVE_ALG_CGM if alg == "cgm" else ms.MSOLVE_ALG_BICGSTABM
    bs = [torch.from_numpy(W.unit_rhs(100 + i, w.n)).pin_memory() for i in range(5)]
    singles = [ms.msolve_solve_host(A, code, b, w.shifts, w.tol, 500) for b in bs]
    singles = [(r.x.clone(), r.iterations, r.conv_iter.copy(), r.relres.copy()) for r in singles]
    batch = ms.msolve_solve_host_batch(A, code, bs, w.shifts, w.tol, 500)
    assert len(batch) == 5
    for r, (x, it, conv, rel) in zip(batch, singles):
        assert r.status == 0 and r.iterations == it and torch.equal(r.x, x)
        assert np.array_equal(r.conv_iter, conv) and np.array_equal(r.relres, rel)
    assert not torch.equal(batch[0].x, batch[1].x)                    # different right-hand sides
    o = oracle_solve(w, np.complex128)                                 # and one of them against the oracle
    w2 = W.config2(extents=(8, 6, 4, 6)) if alg == "cgm" else W.config3(extents=(6, 6, 4, 6))
    w2.b = bs[3].numpy()
    o = oracle_solve(w2, np.complex128)
    g = (0, batch[3].iterations, batch[3].x.numpy(), batch[3].conv_iter, batch[3].relres, 0)
    check_parity(w2, np.complex128, g, o, w2.tol)
    assert ms.msolve_solve_host_batch(A, code, [], w.shifts, w.tol, 500) == []
    ms.msolve_destroy(A)


# ------------------------------------------------------------------------------- deferred multishift update
DEFER_CASES = [("c1", "csr", np.complex128, 1e-10), ("c2", "bsr3", np.complex128, 1e-10), ("c2", "csr", np.complex64, 1e-5),
               ("c2", "lat", np.complex128, 1e-10), ("c5", "csrvector", np.complex128, 1e-10), ("c5", "csrvector", np.complex64, 1e-5)]


def _defer_workload(which):
    return {"c1": W.config1, "c2": W.config2, "c5": lambda: W.config5(n=(1 << 14) + 13)}[which]()


@pytest.mark.parametrize("defer", [1, 3, 7, 16, 32])
@pytest.mark.parametrize("which,fmt,dtype,tol", DEFER_CASES)
def test_deferred_update_matches_oracle_and_stepwise(ms, which, fmt, dtype, tol, defer):
    # MSOLVE_CFG_DEFER_UPDATE = M: p_k, x_k formed once per M iterations from the residuals of the chunk.  Scalars and
    # residuals are those of the step-by-step form (up to the grouping of the |r|^2 partial sums: another grid), so
    # iteration counts, conv_iter and relres agree; x_k against the oracle at the usual bar, and against the
    # step-by-step GPU result
    w = _defer_workload(which)
    g = gpu_solve(ms, w, dtype, fmt, tol=tol, cfg={ms.MSOLVE_CFG_DEFER_UPDATE: defer})
    o = oracle_solve(w, dtype, tol=tol)
    check_parity(w, dtype, g, o, tol)
    g0 = gpu_solve(ms, w, dtype, fmt, tol=tol, cfg={ms.MSOLVE_CFG_DEFER_UPDATE: 0})
    assert abs(g[1] - g0[1]) <= 1 and np.all(np.abs(g[3] - g0[3]) <= 1)
    if g[1] == g0[1] and np.array_equal(g[3], g0[3]):
        assert np.allclose(g[4], g0[4], rtol=1e-9 if dtype == np.complex128 else 1e-3, atol=0)
    assert g0[5] == 2 + 5 * g0[1] and g[5] == 2 + 6 * g[1]
    for k in range(w.shifts.size):
        d = np.linalg.norm(g[2][k].astype(np.complex128) - g0[2][k]) / np.linalg.norm(g0[2][k])
        assert d <= REL[dtype], (k, d)      # two groupings of the |r|^2 sums, amplified by the iteration (as fused vs graph)


@pytest.mark.parametrize("defer", [3, 32])
@pytest.mark.parametrize("max_iter", [1, 2, 3, 4, 7])
def test_deferred_update_when_the_solve_ends_inside_a_chunk(ms, defer, max_iter):
    # MAXITER after max_iter iterations: the pending residuals are flushed, x_k = the iterate of that iteration
    w = W.config2()
    g = gpu_solve(ms, w, np.complex128, "bsr3", max_iter=max_iter, cfg={ms.MSOLVE_CFG_DEFER_UPDATE: defer})
    g0 = gpu_solve(ms, w, np.complex128, "bsr3", max_iter=max_iter, cfg={ms.MSOLVE_CFG_DEFER_UPDATE: 0})
    o = oracle_solve(w, np.complex128, max_iter=max_iter)
    assert g[0] == g0[0] == o.status == oracle.MAXITER and g[1] == g0[1] == max_iter
    for k in range(w.shifts.size):
        assert np.linalg.norm(g[2][k] - o.x[k]) <= 1e-12 * np.linalg.norm(o.x[k]), k
        assert np.linalg.norm(g[2][k] - g0[2][k]) <= 1e-12 * np.linalg.norm(g0[2][k]), k


def test_deferred_update_shifts_that_stop_in_different_chunks(ms):
    # shifts spread over six decades stop far apart (conv_iter from a few iterations to ~100): every x_k is frozen
    # at its own iteration although it is only formed at the next flush; literal stop rule as well
    w = W.config2()
    w.shifts = np.array([0.0, 0.01, 0.1, 1.0, 10.0, 100.0, 1e3, 1e4])
    for rule in (0, 1):
        cfg = {ms.MSOLVE_CFG_DEFER_UPDATE: 5, ms.MSOLVE_CFG_STOP_RULE: rule}
        g = gpu_solve(ms, w, np.complex128, "bsr3", cfg=cfg)
        o = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, w.tol, w.max_iter, stop_rule=rule)
        assert g[0] == o.status == 0 and g[1] == o.iterations and np.array_equal(g[3], o.conv_iter)
        if rule == 0:
            assert len(set(g[3].tolist())) >= 4                          # they do stop at different iterations
        for k in range(w.shifts.size):
            assert np.linalg.norm(g[2][k] - o.x[k]) <= 1e-9 * np.linalg.norm(o.x[k]), (rule, k)


# ------------------------------------------------------------------------------- determinism under repetition
@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
@pytest.mark.parametrize("fmt", ["csrtile", "csrmerge", "csrvector", "bsr3", "lat"])
def test_repeated_launches_bit_identical(ms, fmt, dtype, tol):
    # every reduction has a fixed order and every mbarrier ring a fixed hand-over, so 60 SpMVs and 6 whole
    # solves in a row must return the same bytes (a race or a stale stage would show up as a differing run)
    w = W.config4(extents=(16, 16, 8, 12), tol=tol)
    A = make_matrix(ms, w, dtype, fmt)
    rng = np.random.default_rng(23)
    x = dev((rng.standard_normal(w.n) + 1j * rng.standard_normal(w.n)).astype(dtype))
    y0, d0 = ms.msolve_spmv(A, x)
    y0 = y0.clone()
    for _ in range(60):
        y, d = ms.msolve_spmv(A, x)
        assert d == d0 and torch.equal(y, y0)
    b = dev(w.b.astype(dtype))
    r0 = ms.msolve_cgm(A, b, w.shifts, tol, w.max_iter)
    x0 = r0.x.clone()
    for _ in range(6):
        r = ms.msolve_cgm(A, b, w.shifts, tol, w.max_iter)
        assert r.iterations == r0.iterations and torch.equal(r.x, x0)
    ms.msolve_destroy(A)
