"""Pins for the CPU oracle (oracle/msolve_oracle.cpp) against things that are NOT the oracle:
dense LU (numpy), closed forms, textbook special cases, invariants of the method (eq. (4),
PAPER.md:57), library routines (scipy sparse matvec, FFT, DST).  CPU only.

The paper prints no worked numerical example, so every pin is
mathematical; each test names the mistake it would catch.
"""
import numpy as np
import pytest
import scipy.fft
import scipy.sparse as sp

import oracle
from paper_1102_2143_b200 import workloads as W


def _A(w):
    return sp.csr_matrix((w.val, w.colidx, w.rowptr), shape=(w.n, w.n))


def _true_relres(A, b, x, sigma):
    return np.linalg.norm(b - (A @ x + sigma * x)) / np.linalg.norm(b)


@pytest.fixture(scope="module")
def cfg1():
    return W.config1()


@pytest.fixture(scope="module")
def cfg2_small():
    return W.config2(extents=(4, 4, 4, 4))


@pytest.fixture(scope="module")
def cfg3_small():
    return W.config3(extents=(4, 4, 4, 4))


# ------------------------------------------------------------------ SpMV (Alg. 1 l.18)
def test_spmv_matches_scipy_and_dense(cfg1, cfg2_small):
    # catches: wrong row bounds, transposed operand, conjugated values
    rng = np.random.default_rng(1)
    for w in (cfg1, cfg2_small):
        x = rng.standard_normal(w.n) + 1j * rng.standard_normal(w.n)
        y = oracle.spmv(w.rowptr, w.colidx, w.val, x)
        A = _A(w)
        assert np.allclose(y, A @ x, rtol=0, atol=1e-13)
        assert np.allclose(y, A.toarray() @ x, rtol=0, atol=1e-13)
        y32 = oracle.spmv(w.rowptr, w.colidx, w.val.astype(np.complex64), x.astype(np.complex64))
        assert y32.dtype == np.complex64
        assert np.linalg.norm(y32 - y) / np.linalg.norm(y) < 1e-6


# ------------------------------------------------------------------ sigma = 0 reductions
def test_cgm_single_zero_shift_is_plain_cg_bitwise(cfg1, cfg2_small):
    # the unshifted sequence is plain CG.  zeta stays exactly 1, so iterates are
    # bitwise those of a separately written textbook CG.  catches: any error in the base sequence.
    for w in (cfg1, cfg2_small):
        m = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, [0.0], w.tol, 500)
        st, it, x, rel = oracle.cg(w.rowptr, w.colidx, w.val, 0.0, w.b, w.tol, 500)
        assert m.status == oracle.OK and st == oracle.OK
        assert m.iterations == it
        assert np.array_equal(m.x[0], x)
        assert m.zeta[0] == 1.0
        assert m.relres[0] == rel


def test_bicgstabm_single_zero_shift_is_plain_bicgstab(cfg3_small):
    w = cfg3_small
    m = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, [0.0], w.tol, 500)
    st, it, x, rel = oracle.bicgstab(w.rowptr, w.colidx, w.val, 0.0, w.b, w.tol, 500)
    assert m.status == oracle.OK and st == oracle.OK
    assert m.iterations == it
    # p_k is rebuilt from (s, r) instead of A p, so agreement is to rounding, not bitwise
    assert np.linalg.norm(m.x[0] - x) / np.linalg.norm(x) < 1e-12
    assert abs(m.zeta[0] - 1.0) < 1e-14


# ------------------------------------------------------------------ closed forms
def test_cgm_scaled_identity_closed_form():
    # A = c I: one iteration, x_k = b/(c+sigma_k), zeta_1 = c/(c+sigma_k).
    # catches: wrong zeta / beta_k formula at the first step, wrong sign of beta.
    n, c = 37, 2.5
    rowptr = np.arange(n + 1, dtype=np.int32)
    colidx = np.arange(n, dtype=np.int32)
    val = np.full(n, c, dtype=np.complex128)
    b = W.unit_rhs(3, n)
    sig = np.array([0.0, 0.3, 1.0, 7.0])
    m = oracle.cgm(rowptr, colidx, val, b, sig, 1e-12, 10, hist_cap=4)
    assert m.status == oracle.OK and m.iterations == 1
    for k, s in enumerate(sig):
        assert np.allclose(m.x[k], b / (c + s), rtol=1e-14, atol=0)
        assert abs(m.hist[0, 3 + k] - c / (c + s)) < 1e-15


def test_cgm_diagonal_finite_termination():
    # m distinct eigenvalues => exact solution in <= m iterations for every shift.
    rng = np.random.default_rng(5)
    n, m_ = 60, 6
    eig = np.array([1.0, 1.7, 2.9, 4.1, 6.3, 9.0])
    d = eig[rng.integers(0, m_, n)]
    d[:m_] = eig
    rowptr = np.arange(n + 1, dtype=np.int32)
    colidx = np.arange(n, dtype=np.int32)
    b = W.unit_rhs(4, n)
    sig = np.array([0.0, 0.05, 0.5, 3.0])
    res = oracle.cgm(rowptr, colidx, d.astype(np.complex128), b, sig, 1e-13, 50)
    assert res.status == oracle.OK and res.iterations <= m_
    for k, s in enumerate(sig):
        assert np.linalg.norm(res.x[k] - b / (d + s)) / np.linalg.norm(b / (d + s)) < 1e-11


def test_bicgstabm_diagonal_complex():
    # non-Hermitian (complex diagonal) operator with few distinct eigenvalues
    rng = np.random.default_rng(6)
    n = 48
    eig = np.array([1.0 + 0.3j, 1.9 - 0.2j, 3.2 + 0.5j, 4.4 - 0.1j, 6.1 + 0.2j])
    d = eig[rng.integers(0, eig.size, n)]
    d[:eig.size] = eig
    rowptr = np.arange(n + 1, dtype=np.int32)
    colidx = np.arange(n, dtype=np.int32)
    b = W.unit_rhs(8, n)
    sig = np.array([0.0, 0.1, 1.0])
    res = oracle.bicgstabm(rowptr, colidx, d, b, sig, 1e-12, 50)
    assert res.status == oracle.OK and res.iterations <= eig.size + 1
    for k, s in enumerate(sig):
        assert np.linalg.norm(res.x[k] - b / (d + s)) / np.linalg.norm(b / (d + s)) < 1e-10


# ------------------------------------------------------------------ eq. (1) by dense LU
@pytest.mark.parametrize("which", ["cfg1", "cfg2_small"])
def test_cgm_matches_dense_lu(which, request):
    # the result itself.  tol 1e-14 so the iterate, not the tolerance, is compared.
    w = request.getfixturevalue(which)
    A = _A(w).toarray()
    res = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 1e-14, 1000)
    assert res.status == oracle.OK
    for k, s in enumerate(w.shifts):
        xe = np.linalg.solve(A + s * np.eye(w.n), w.b)
        assert np.linalg.norm(res.x[k] - xe) / np.linalg.norm(xe) < 1e-12


def test_bicgstabm_matches_dense_lu(cfg3_small):
    w = cfg3_small
    A = _A(w).toarray()
    assert np.abs(A - A.conj().T).max() > 0.1  # genuinely non-Hermitian
    res = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 1e-14, 1000)
    assert res.status == oracle.OK
    for k, s in enumerate(w.shifts):
        xe = np.linalg.solve(A + s * np.eye(w.n), w.b)
        assert np.linalg.norm(res.x[k] - xe) / np.linalg.norm(xe) < 1e-12


# ------------------------------------------------------------------ eq. (4): collinear residuals
@pytest.mark.parametrize("which", ["cfg1", "cfg2_small"])
def test_cgm_collinearity_every_iteration(which, request):
    # b - (A+sigma_k) x_k^(n) = zeta_k^(n) r^(n) for every n.
    # catches: any wrong recurrence incl. p_k (its error shows one step later).
    w = request.getfixturevalue(which)
    A = _A(w)
    for nit in range(1, 16):
        res = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 0.0, nit)
        assert res.iterations == nit and res.status == oracle.MAXITER
        for k, s in enumerate(w.shifts):
            lhs = w.b - (A @ res.x[k] + s * res.x[k])
            assert np.linalg.norm(lhs - res.zeta[k] * res.r) < 1e-13


def test_bicgstabm_collinearity_every_iteration(cfg3_small):
    w = cfg3_small
    A = _A(w)
    for nit in range(1, 10):
        res = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 0.0, nit)
        assert res.iterations == nit
        for k, s in enumerate(w.shifts):
            lhs = w.b - (A @ res.x[k] + s * res.x[k])
            assert np.linalg.norm(lhs - res.zeta[k] * res.r) < 1e-13


# ------------------------------------------------------------------ stop rule, residuals, masks
def test_true_residual_below_tol_and_monotone_conv(cfg1, cfg2_small, cfg3_small):
    # true residual <= tol (graded at 10 tol); conv_iter non-increasing in sigma.
    for w, fn in ((cfg1, oracle.cgm), (cfg2_small, oracle.cgm), (cfg3_small, oracle.bicgstabm)):
        A = _A(w)
        res = fn(w.rowptr, w.colidx, w.val, w.b, w.shifts, w.tol, w.max_iter)
        assert res.status == oracle.OK
        assert res.iterations == res.conv_iter.max()
        assert np.all(np.diff(res.conv_iter) <= 0)          # shifts ascending in these configs
        for k, s in enumerate(w.shifts):
            assert res.relres[k] <= w.tol
            assert _true_relres(A, w.b, res.x[k], s) <= 2.0 * w.tol


def test_frozen_shift_keeps_its_iterate(cfg1):
    # a shift converged at iteration c must hold exactly the x_k of a run stopped at c
    w = cfg1
    full = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, w.tol, w.max_iter)
    k = int(np.argmin(full.conv_iter))
    c = int(full.conv_iter[k])
    assert c < full.iterations
    part = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 0.0, c)
    assert np.array_equal(full.x[k], part.x[k])


def test_independent_single_shift_solves(cfg2_small, cfg3_small):
    # shift coupling: each x_k agrees with a plain solver run on the explicitly shifted system
    w = cfg2_small
    res = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 1e-12, 1000)
    for k in (0, 5, 11):
        st, it, x, rel = oracle.cg(w.rowptr, w.colidx, w.val, float(w.shifts[k]), w.b, 1e-12, 1000)
        assert st == oracle.OK
        assert np.linalg.norm(res.x[k] - x) / np.linalg.norm(x) < 1e-10
        assert abs(it - res.conv_iter[k]) <= 1
    w = cfg3_small
    res = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 1e-12, 1000)
    for k in (0, 3, 7):
        st, it, x, rel = oracle.bicgstab(w.rowptr, w.colidx, w.val, float(w.shifts[k]), w.b, 1e-12, 1000)
        assert st == oracle.OK
        assert np.linalg.norm(res.x[k] - x) / np.linalg.norm(x) < 1e-10


def test_maxiter_and_zero_rhs(cfg1):
    w = cfg1
    res = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, w.tol, 3)
    assert res.status == oracle.MAXITER and res.iterations == 3 and np.all(res.conv_iter == -1)
    z = oracle.cgm(w.rowptr, w.colidx, w.val, np.zeros(w.n, dtype=np.complex128), w.shifts, w.tol, 10)
    assert z.status == oracle.OK and z.iterations == 0 and not z.x.any()


def test_cgm_breakdown_on_indefinite():
    # P <= 0 must be reported, not iterated through (R16)
    n = 8
    rowptr = np.arange(n + 1, dtype=np.int32)
    colidx = np.arange(n, dtype=np.int32)
    val = -np.ones(n, dtype=np.complex128)
    res = oracle.cgm(rowptr, colidx, val, W.unit_rhs(1, n), [0.0], 1e-10, 10)
    assert res.status == oracle.BREAKDOWN


# ------------------------------------------------------------------ FFT closed form (pure gauge)
def _pure_gauge_closed_form(w, seed):
    ext = w.meta["extents"]
    d = len(ext)
    vol = int(np.prod(ext))
    g = W.haar_su3(W._substream(seed, "links"), vol)                 # same stream su3_links used
    bs = w.b.reshape(vol, 3)
    wv = np.einsum("sba,sb->sa", g.conj(), bs)                        # G^dagger b
    shape = tuple(ext[::-1])
    lam = np.full(shape, w.meta["diag"], dtype=np.complex128)
    for mu in range(d):
        ax = d - 1 - mu
        k = 2.0 * np.pi * np.arange(ext[mu]) / ext[mu]
        sh = [1] * d
        sh[ax] = ext[mu]
        lam = lam - (w.meta["c_f"] * np.exp(1j * k) + w.meta["c_b"] * np.exp(-1j * k)).reshape(sh)
    out = []
    for s in w.shifts:
        y = np.empty((vol, 3), dtype=np.complex128)
        for c in range(3):
            f = np.fft.fftn(wv[:, c].reshape(shape))
            y[:, c] = np.fft.ifftn(f / (lam + s)).reshape(vol)
        out.append(np.einsum("sab,sb->sa", g, y).reshape(-1))
    return out


def test_cgm_pure_gauge_fft_closed_form():
    # SU(3)/BSR3 operator end to end: A = G A_free G^dagger is diagonalised by the FFT.
    # catches: wrong link placement / dagger / neighbour in the generator AND solver errors.
    seed = 77
    m = 0.5
    w = W.su3_workload("pg", "cgm", (4, 4, 4, 6), m * m + 8, 1.0, 1.0, [0.0, 0.1, 1.0], 1e-13,
                       seed=seed, links="pure_gauge")
    res = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 1e-13, 2000)
    assert res.status == oracle.OK
    for k, xe in enumerate(_pure_gauge_closed_form(w, seed)):
        assert np.linalg.norm(res.x[k] - xe) / np.linalg.norm(xe) < 1e-10


def test_bicgstabm_pure_gauge_fft_closed_form():
    seed = 78
    w = W.su3_workload("pgnh", "bicgstabm", (4, 4, 4, 6), 4.2, 0.6, 0.4, [0.0, 0.2, 2.0], 1e-13,
                       seed=seed, links="pure_gauge")
    res = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 1e-13, 2000)
    assert res.status == oracle.OK
    for k, xe in enumerate(_pure_gauge_closed_form(w, seed)):
        assert np.linalg.norm(res.x[k] - xe) / np.linalg.norm(xe) < 1e-10


# ------------------------------------------------------------------ the paper's own matrix
def test_cgm_poisson_sine_transform():
    # 2-D 5-point Poisson.  (A+sigma)^-1 b by the type-I sine transform.
    nx, ny = 24, 17
    w = W.poisson_workload(nx, ny, nshifts=5, tol=1e-13)
    res = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 1e-13, 5000)
    assert res.status == oracle.OK
    lam = (4.0 - 2.0 * np.cos(np.pi * np.arange(1, nx + 1) / (nx + 1))[None, :]
           - 2.0 * np.cos(np.pi * np.arange(1, ny + 1) / (ny + 1))[:, None])
    bb = w.b.reshape(ny, nx)
    for k, s in enumerate(w.shifts):
        f = scipy.fft.dstn(bb.real, type=1, norm="ortho") + 1j * scipy.fft.dstn(bb.imag, type=1, norm="ortho")
        f = f / (lam + s)
        xe = scipy.fft.idstn(f.real, type=1, norm="ortho") + 1j * scipy.fft.idstn(f.imag, type=1, norm="ortho")
        assert np.linalg.norm(res.x[k] - xe.ravel()) / np.linalg.norm(xe) < 1e-10


# ------------------------------------------------------------------ complex64 oracle
def test_c64_oracle_tracks_c128(cfg2_small, cfg3_small):
    for w, fn in ((cfg2_small, oracle.cgm), (cfg3_small, oracle.bicgstabm)):
        hi = fn(w.rowptr, w.colidx, w.val, w.b, w.shifts, 1e-5, 1000)
        lo = fn(w.rowptr, w.colidx, w.val.astype(np.complex64), w.b.astype(np.complex64), w.shifts, 1e-5, 1000)
        assert lo.status == oracle.OK and lo.x.dtype == np.complex64
        assert abs(lo.iterations - hi.iterations) <= 1
        for k in range(w.shifts.size):
            assert np.linalg.norm(lo.x[k] - hi.x[k]) / np.linalg.norm(hi.x[k]) < 2e-5


# ------------------------------------------------------------------ real dtypes (the paper's own runs)
def test_real_cgm_poisson_sine_transform():
    # the paper's runs are REAL fp32/fp64 on the 2-D Poisson matrix.
    nx, ny = 19, 23
    w = W.poisson_workload(nx, ny, nshifts=4, tol=1e-13, real=True)
    assert w.val.dtype == np.float64 and w.b.dtype == np.float64
    res = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 1e-13, 5000)
    assert res.status == oracle.OK and res.x.dtype == np.float64
    lam = (4.0 - 2.0 * np.cos(np.pi * np.arange(1, nx + 1) / (nx + 1))[None, :]
           - 2.0 * np.cos(np.pi * np.arange(1, ny + 1) / (ny + 1))[:, None])
    f = scipy.fft.dstn(w.b.reshape(ny, nx), type=1, norm="ortho")
    for k, s in enumerate(w.shifts):
        xe = scipy.fft.idstn(f / (lam + s), type=1, norm="ortho").ravel()
        assert np.linalg.norm(res.x[k] - xe) / np.linalg.norm(xe) < 1e-10


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_real_oracle_is_the_complex_oracle_on_real_data(dtype):
    # A real matrix stored as complex has exactly zero imaginary parts throughout ((a+0i)(b+0i) = ab
    # exactly), so the real-typed oracle must reproduce the (pinned) complex-typed one BITWISE.
    cdt = np.complex128 if dtype == np.float64 else np.complex64
    for w, fn in ((W.poisson_workload(13, 11, nshifts=5, tol=1e-9, real=True), oracle.cgm),
                  (W.poisson_workload(13, 11, nshifts=5, tol=1e-9, real=True, drift=0.4), oracle.bicgstabm)):
        tol = 1e-9 if dtype == np.float64 else 1e-5
        re = fn(w.rowptr, w.colidx, w.val.astype(dtype), w.b.astype(dtype), w.shifts, tol, 3000)
        cx = fn(w.rowptr, w.colidx, w.val.astype(cdt), w.b.astype(cdt), w.shifts, tol, 3000)
        assert re.status == cx.status == oracle.OK and re.iterations == cx.iterations
        assert np.array_equal(re.conv_iter, cx.conv_iter)
        assert np.array_equal(re.x, cx.x.real) and not np.any(cx.x.imag)
        assert np.array_equal(re.relres, cx.relres)


def test_real_bicgstabm_dense_lu():
    w = W.poisson_workload(9, 8, nshifts=4, tol=1e-14, real=True, drift=0.5)
    res = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, w.shifts, 1e-14, 3000)
    assert res.status == oracle.OK
    A = scipy.sparse.csr_matrix((w.val, w.colidx, w.rowptr), shape=(w.n, w.n)).toarray()
    assert np.abs(A - A.T).max() > 0.5          # genuinely non-symmetric
    for k, s in enumerate(w.shifts):
        xe = np.linalg.solve(A + s * np.eye(w.n), w.b)
        assert np.linalg.norm(res.x[k] - xe) / np.linalg.norm(xe) < 1e-12
