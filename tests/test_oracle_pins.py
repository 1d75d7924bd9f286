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


# ------------------------------------------------------------------ stop_rule = 1 (Alg. 1 l.15 read literally)
def test_stop_rule_base_cgm(cfg1, cfg2_small):
    # "while |r| > eps" on the UNSHIFTED system.  Pins: (a) the base Krylov sequence does not
    # depend on the shifts, so the loop runs exactly as long as textbook CG on A (same R1 bitwise, same test);
    # (b) with sigma = 0 among the shifts the default rule ends at the same iteration (zeta_0 = 1) with the
    # same bits in x_0; (c) the other shifts are NOT frozen: they keep converging, so their true residual is
    # no larger than under the default rule and every conv_iter equals the exit iteration.
    # catches: testing |zeta_k| |r| instead of |r|, freezing shifts early, wrong exit bookkeeping.
    for w in (cfg1, cfg2_small):
        A = _A(w)
        sig = np.array([0.37, 0.011, 2.0])                               # sigma = 0 NOT among them
        st, it, _, rel = oracle.cg(w.rowptr, w.colidx, w.val, 0.0, w.b, w.tol, 500)
        m1 = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, sig, w.tol, 500, stop_rule=1)
        m0 = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, sig, w.tol, 500, stop_rule=0)
        assert st == oracle.OK and m1.status == oracle.OK
        assert m1.iterations == it and np.all(m1.conv_iter == it)
        assert m0.iterations <= it and m0.conv_iter[2] < it              # under the default rule sigma = 2 stops early
        for k, s in enumerate(sig):
            assert abs(m1.relres[k] - abs(m1.zeta[k]) * rel) <= 1e-14 * m1.relres[k]   # reported: |zeta_k| ||r|| / ||b|| at exit
            assert _true_relres(A, w.b, m1.x[k], s) <= _true_relres(A, w.b, m0.x[k], s) * (1 + 1e-6)
            assert _true_relres(A, w.b, m1.x[k], s) <= w.tol
        sig0 = np.array([0.0, 0.37, 2.0])                                # sigma = 0 among them
        a = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, sig0, w.tol, 500, stop_rule=1)
        b = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, sig0, w.tol, 500, stop_rule=0)
        assert a.iterations == b.iterations == it and np.array_equal(a.x[0], b.x[0])
        assert np.all(a.conv_iter == it) and b.conv_iter[2] < it
        # max_iter reached first: MAXITER, nothing converged
        c = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, sig0, w.tol, 3, stop_rule=1)
        assert c.status == oracle.MAXITER and c.iterations == 3 and np.all(c.conv_iter == -1)


def test_stop_rule_base_bicgstabm(cfg3_small):
    # the same for BiCGStab-M against textbook BiCGStab on the unshifted matrix
    w = cfg3_small
    A = _A(w)
    sig = np.array([0.3, 0.05, 1.5])
    st, it, _, rel = oracle.bicgstab(w.rowptr, w.colidx, w.val, 0.0, w.b, w.tol, 500)
    m1 = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, sig, w.tol, 500, stop_rule=1)
    m0 = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, sig, w.tol, 500, stop_rule=0)
    assert st == oracle.OK and m1.status == oracle.OK
    assert m1.iterations == it and np.all(m1.conv_iter == it) and m0.iterations <= it
    for k, s in enumerate(sig):
        assert abs(m1.relres[k] - abs(m1.zeta[k]) * rel) <= 1e-9 * m1.relres[k]
        assert _true_relres(A, w.b, m1.x[k], s) <= 10 * w.tol
    a = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, np.array([0.0, 0.3]), w.tol, 500, stop_rule=1)
    b = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, np.array([0.0, 0.3]), w.tol, 500, stop_rule=0)
    assert a.iterations == b.iterations and np.array_equal(a.x[0], b.x[0])


# ------------------------------------------------------------------ the per-iteration scalar history
def _textbook_bicgstab_scalars(M, b, nit):
    """van der Vorst's BiCGStab on the dense matrix M in numpy, shadow vector b: per iteration
    (alpha, omega, beta, ||r||^2).  An independent restatement of the textbook, not of the oracle."""
    r = b.copy(); p = b.copy(); rhat = b.copy()
    rho = np.vdot(rhat, r)
    out = []
    for _ in range(nit):
        v = M @ p
        a = rho / np.vdot(rhat, v)
        s = r - a * v
        t = M @ s
        om = np.vdot(t, s) / np.vdot(t, t)
        r = s - om * t
        rho_new = np.vdot(rhat, r)
        bt = (rho_new / rho) * (a / om)
        p = r + bt * (p - om * v)
        rho = rho_new
        out.append((a, om, bt, np.vdot(r, r).real, r.copy()))
    return out


def test_bicgstabm_history_against_textbook_and_true_residuals(cfg3_small):
    # Base row = textbook BiCGStab on A: beta = -alpha, chi = omega, alpha' = textbook beta, |r'|^2.
    # Per shift: beta_k = -(the BiCG step length of the system A + sigma_k I), which textbook BiCGStab on the
    # shifted matrix recovers whatever its own omega is; chi_k and zeta_new through the shifted residual
    # b - (A + sigma_k) x_k (numpy, from the iterate) whose norm must equal |zeta_k rho_k| ||r|| with
    # rho_k = prod_j chi_k[j] / chi[j] (rho' = rho / (1 + chi sigma) = rho chi_k / chi).
    # catches: a wrong zeta / beta_k / chi_k / rho recurrence, a wrong slot in the history row.
    w = cfg3_small
    A = _A(w)
    M = A.toarray()
    sig = np.array([0.0, 0.2, 1.0])
    nit, S = 6, 3
    m = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, sig, 0.0, nit, hist_cap=nit)
    assert m.hist.shape == (nit, 8 + 6 * S)
    base = _textbook_bicgstab_scalars(M, w.b, nit)
    per_shift = [_textbook_bicgstab_scalars(M + s * np.eye(w.n), w.b, nit) for s in sig]
    rho = np.ones(S, dtype=np.complex128)
    for n in range(nit):
        h = m.hist[n]
        beta, chi, alpha_new = h[0] + 1j * h[1], h[2] + 1j * h[3], h[4] + 1j * h[5]
        a, om, bt, rr, _ = base[n]
        assert abs(beta + a) <= 1e-10 * abs(a) and abs(chi - om) <= 1e-10 * abs(om)
        assert abs(alpha_new - bt) <= 1e-9 * abs(bt) and abs(h[6] - rr) <= 1e-9 * rr and h[7] == 0.0
        zeta_new = h[8:8 + 2 * S].view(np.complex128)
        beta_k = h[8 + 2 * S:8 + 4 * S].view(np.complex128)
        chi_k = h[8 + 4 * S:8 + 6 * S].view(np.complex128)
        rho = rho * chi_k / chi
        xn = oracle.bicgstabm(w.rowptr, w.colidx, w.val, w.b, sig, 0.0, n + 1).x
        for k in range(S):
            ak = per_shift[k][n][0]
            assert abs(beta_k[k] + ak) <= 1e-8 * abs(ak), (n, k)
            tr = np.linalg.norm(w.b - (A @ xn[k] + sig[k] * xn[k]))
            assert abs(abs(zeta_new[k] * rho[k]) * np.sqrt(rr) - tr) <= 1e-8 * tr, (n, k)
        assert abs(zeta_new[0] - 1.0) < 1e-13 and abs(chi_k[0] - chi) == 0.0   # sigma = 0: the base system itself


def test_cgm_history_is_the_shifted_systems_own_cg(cfg2_small):
    # CG-M: beta_k = -(textbook CG step length on A + sigma_k I), alpha_k = its direction coefficient,
    # |zeta_k| = ||r^sigma|| / ||r||; base row: beta = -step length of CG on A, alpha_next = R1/R0, R1.
    w = cfg2_small
    M = _A(w).toarray()
    sig = np.array([0.0, 0.3, 2.0])
    nit, S = 7, 3
    m = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, sig, 0.0, nit, hist_cap=nit)
    assert m.hist.shape == (nit, 3 + 3 * S)

    def textbook_cg(Mk):
        r = w.b.copy(); p = w.b.copy(); rr = np.vdot(r, r).real
        out = []
        for _ in range(nit):
            q = Mk @ p
            a = rr / np.vdot(p, q).real
            r = r - a * q
            rr_new = np.vdot(r, r).real
            bt = rr_new / rr
            p = r + bt * p
            rr = rr_new
            out.append((a, bt, rr))
        return out

    base = textbook_cg(M)
    shifted = [textbook_cg(M + s * np.eye(w.n)) for s in sig]
    for n in range(nit):
        h = m.hist[n]
        a, bt, rr = base[n]
        assert abs(h[0] + a) <= 1e-11 * a and abs(h[1] - bt) <= 1e-10 * bt and abs(h[2] - rr) <= 1e-10 * rr
        for k in range(S):
            ak, btk, rrk = shifted[k][n]
            assert abs(h[3 + S + k] + ak) <= 1e-10 * ak, (n, k)                      # beta_k
            assert abs(h[3 + 2 * S + k] - btk) <= 1e-9 * btk, (n, k)                 # alpha_k
            assert abs(abs(h[3 + k]) - np.sqrt(rrk / rr)) <= 1e-9 * np.sqrt(rrk / rr), (n, k)   # zeta_new


# ------------------------------------------------------------------ eq. (6): a right-hand side per shift
@pytest.mark.parametrize("alg", ["cgm", "bicgstabm"])
def test_multirhs_matches_dense_lu_and_common_residual(alg, cfg2_small, cfg3_small):
    # PAPER.md:228-232.  Pins: (a) the initial guesses really give ONE residual: b_i - (A + sigma_i) y_i = r0 for
    # every i (numpy, from the returned y and r0); (b) each x_i against a dense LU solve of (A + sigma_i) x = b_i;
    # (c) the true residual of every system is below tol relative to ITS right-hand side.
    # catches: wrong divided differences, a wrong sigma in the u recursion, wrong Newton weights in y_i, x_i = z_i.
    w = cfg2_small if alg == "cgm" else cfg3_small
    A = _A(w)
    M = A.toarray()
    sig = np.array([0.0, 0.35, 1.1, 2.0])
    rng = np.random.default_rng(8)
    B = rng.standard_normal((sig.size, w.n)) + 1j * rng.standard_normal((sig.size, w.n))
    B /= np.linalg.norm(B, axis=1)[:, None]
    B[2] *= 3.0                                            # different norms: the thresholds are per system
    r = oracle.multirhs(w.rowptr, w.colidx, w.val, B, sig, 1e-13, 500, alg)
    assert r.status == oracle.OK
    for i, s in enumerate(sig):
        assert np.linalg.norm(B[i] - (A @ r.y[i] + s * r.y[i]) - r.r0) <= 1e-12 * np.linalg.norm(r.r0), i
        x_lu = np.linalg.solve(M + s * np.eye(w.n), B[i])
        assert np.linalg.norm(r.x[i] - x_lu) / np.linalg.norm(x_lu) < 1e-10, i
        assert np.linalg.norm(B[i] - (A @ r.x[i] + s * r.x[i])) <= 1e-11 * np.linalg.norm(B[i]), i
    # at a loose tolerance every system stops by its own norm: true residual <= tol ||b_i|| (<= 10 tol graded)
    r = oracle.multirhs(w.rowptr, w.colidx, w.val, B, sig, 1e-8, 500, alg)
    for i, s in enumerate(sig):
        assert r.relres[i] <= 1e-8
        assert np.linalg.norm(B[i] - (A @ r.x[i] + s * r.x[i])) <= 1e-7 * np.linalg.norm(B[i]), i


def test_multirhs_special_cases(cfg2_small):
    w = cfg2_small
    rng = np.random.default_rng(9)
    # two systems: the closed form y_0 = y_1 = (b_1 - b_0) / (sigma_1 - sigma_0), r0 = b_0 - (A + sigma_0) y
    sig = np.array([0.2, 0.9])
    B = rng.standard_normal((2, w.n)) + 1j * rng.standard_normal((2, w.n))
    r = oracle.multirhs(w.rowptr, w.colidx, w.val, B, sig, 1e-12, 500)
    y = (B[1] - B[0]) / (sig[1] - sig[0])
    assert np.allclose(r.y[0], y, rtol=1e-14, atol=0) and np.array_equal(r.y[0], r.y[1])
    assert np.allclose(r.r0, B[0] - (_A(w) @ y + sig[0] * y), rtol=0, atol=1e-13 * np.linalg.norm(r.r0))
    # the same right-hand side for every shift IS eq. (1): all divided differences vanish, y = 0, r0 = b, and the
    # result is the plain multishift solve bit for bit
    sig = np.array([0.0, 0.01, 0.3, 1.0])
    B = np.tile(w.b, (4, 1))
    r = oracle.multirhs(w.rowptr, w.colidx, w.val, B, sig, w.tol, 500)
    m = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, sig, w.tol, 500)
    assert not r.y.any() and np.array_equal(r.r0, w.b)
    assert r.iterations == m.iterations and np.array_equal(r.x, m.x) and np.array_equal(r.conv_iter, m.conv_iter)
    # right-hand sides that are a polynomial of degree 2 in the shift: only d_0, d_1, d_2 are non-zero
    c = rng.standard_normal((3, w.n)) + 1j * rng.standard_normal((3, w.n))
    sig = np.array([0.1, 0.5, 0.8, 1.4, 2.2])
    B = np.array([c[0] + s * c[1] + s * s * c[2] for s in sig])
    r = oracle.multirhs(w.rowptr, w.colidx, w.val, B, sig, 1e-12, 500)
    M = _A(w).toarray()
    for i, s in enumerate(sig):
        x_lu = np.linalg.solve(M + s * np.eye(w.n), B[i])
        assert np.linalg.norm(r.x[i] - x_lu) / np.linalg.norm(x_lu) < 1e-10
    # one system: nothing to construct
    r = oracle.multirhs(w.rowptr, w.colidx, w.val, w.b[None, :], [0.3], w.tol, 500)
    m = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, [0.3], w.tol, 500)
    assert np.array_equal(r.x, m.x)
    # duplicate shifts cannot be served by this construction
    with pytest.raises(ValueError):
        oracle.multirhs(w.rowptr, w.colidx, w.val, B[:2], [0.5, 0.5], 1e-10, 10)
