"""GPU parity of msolve_solve_multirhs (a right-hand side per shift, eq. (6); SURVEY.md
8(f)-4) against the oracle's step-by-step construction on the same seeded inputs."""
import numpy as np
import pytest
import scipy.sparse as sp
import torch

import oracle
from paper_1102_2143_b200 import workloads as W
from test_gpu_parity import MAXABS_C, REL, dev, make_matrix, ms  # noqa: F401

pytestmark = pytest.mark.gpu


def _rhs(seed, shifts, n, dtype, noise):
    """b_i = c_0 + sigma_i c_1 + noise * g_i: right-hand sides that vary smoothly with the shift plus an independent
    part.  (The construction extrapolates the interpolant of the b_i from the shifts to -spec(A); with independent
    right-hand sides that factor grows like ||A||^(S-1) / prod |sigma_i - sigma_j|, see include/msolve.h.)"""
    rng = np.random.default_rng(seed)
    c = rng.standard_normal((2, n)) + 1j * rng.standard_normal((2, n))
    g = rng.standard_normal((len(shifts), n)) + 1j * rng.standard_normal((len(shifts), n))
    B = np.array([c[0] + t * c[1] + noise * g[i] for i, t in enumerate(shifts)])
    return (B / np.linalg.norm(B[0])).astype(dtype)


def _compare(ms, w, dtype, tol, shifts, B, g, o, bar, res_bar=None):
    assert g.status == o.status == 0 and abs(g.iterations - o.iterations) <= 2
    assert np.all(np.abs(g.conv_iter - o.conv_iter) <= 2)
    M = sp.csr_matrix((w.val, w.colidx, w.rowptr), shape=(w.n, w.n))
    x = g.x.cpu().numpy()
    for i, s in enumerate(shifts):
        diff = x[i].astype(np.complex128) - o.x[i]
        assert np.linalg.norm(diff) <= bar * np.linalg.norm(o.x[i]), (i, np.linalg.norm(diff) / np.linalg.norm(o.x[i]))
        assert np.abs(diff).max() <= MAXABS_C * bar * np.abs(o.x[i]).max(), i
        xi = x[i].astype(np.complex128)
        bi = B[i].astype(np.complex128)
        assert np.linalg.norm(bi - (M @ xi + s * xi)) <= (res_bar or 10 * tol) * np.linalg.norm(bi), i     # relative to ITS rhs
        assert g.relres[i] <= tol * (1 + 1e-9)


@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
@pytest.mark.parametrize("alg,fmt", [("cgm", "bsr3"), ("cgm", "csr"), ("bicgstabm", "bsr3"), ("cgm", "lat")])
def test_multirhs_matches_oracle(ms, alg, fmt, dtype, tol):
    w = W.config2(extents=(6, 6, 4, 6)) if alg == "cgm" else W.config3(extents=(6, 6, 4, 6))
    code = ms.MSOLVE_ALG_CGM if alg == "cgm" else ms.MSOLVE_ALG_BICGSTABM
    shifts = np.array([0.0, 0.5, 1.3])
    B = _rhs(31, shifts, w.n, dtype, 0.05)
    A = make_matrix(ms, w, dtype, fmt)
    g = ms.msolve_solve_multirhs(A, code, dev(B), shifts, tol, w.max_iter)
    o = oracle.multirhs(w.rowptr, w.colidx, w.val.astype(dtype), B, shifts, tol, w.max_iter, alg)
    _compare(ms, w, dtype, tol, shifts, B, g, o, REL[dtype])
    ms.msolve_destroy(A)


def test_multirhs_independent_rhs_c128(ms):
    # five INDEPENDENT Gaussian right-hand sides of different norms: ||r0|| / ||b|| ~ ||A||^4 here, which complex128
    # still absorbs at tol 1e-10 (complex64 does not: eps ||r0|| > tol ||b||)
    w = W.config2(extents=(6, 6, 4, 6))
    shifts = np.array([0.0, 0.4, 1.0, 1.7, 2.5])
    rng = np.random.default_rng(31)
    B = rng.standard_normal((5, w.n)) + 1j * rng.standard_normal((5, w.n))
    B /= np.linalg.norm(B, axis=1)[:, None]
    B *= np.linspace(1.0, 3.0, 5)[:, None]
    A = make_matrix(ms, w, np.complex128, "bsr3")
    g = ms.msolve_solve_multirhs(A, ms.MSOLVE_ALG_CGM, dev(B), shifts, 1e-10, w.max_iter)
    o = oracle.multirhs(w.rowptr, w.colidx, w.val, B, shifts, 1e-10, w.max_iter)
    _compare(ms, w, np.complex128, 1e-10, shifts, B, g, o, 1e-9)
    ms.msolve_destroy(A)


def test_multirhs_many_shifts(ms):
    # 20 shifts (> 16: the level-by-level divided-difference kernels and the generic guess kernel).  Twenty nodes
    # are only usable where the extrapolation from the shifts to -spec(A) is benign: an operator whose norm is small
    # against the spacing of the shifts (here ||A|| ~ 0.01, shifts 1, 2, ..., 20).
    w = W.config2(extents=(4, 6, 4, 6))
    w.val = w.val * (0.01 / 13.0)
    w.blocks = w.blocks * (0.01 / 13.0)
    shifts = np.arange(1.0, 21.0)
    B = _rhs(32, shifts, w.n, np.complex128, 0.05)
    A = make_matrix(ms, w, np.complex128, "bsr3")
    g = ms.msolve_solve_multirhs(A, ms.MSOLVE_ALG_CGM, dev(B), shifts, 1e-10, w.max_iter)
    o = oracle.multirhs(w.rowptr, w.colidx, w.val, B, shifts, 1e-10, w.max_iter)
    # the guesses carry the rounding of the 20-node extrapolation (binomial weights up to C(20,10) ~ 2e5 times eps), so
    # the true residual floors near 1e-9 ||b_i|| on both sides although the recurrence residual reaches 1e-10
    _compare(ms, w, np.complex128, 1e-10, shifts, B, g, o, 1e-7, res_bar=1e-7)
    ms.msolve_destroy(A)


def test_multirhs_reductions_and_validation(ms):
    w = W.config2(extents=(4, 4, 4, 4))
    A = make_matrix(ms, w, np.complex128, "bsr3")
    shifts = np.array([0.0, 0.01, 0.3, 1.0])
    # the same right-hand side for every shift is eq. (1): the plain multishift solve, bit for bit
    B = np.tile(w.b, (4, 1))
    g = ms.msolve_solve_multirhs(A, ms.MSOLVE_ALG_CGM, dev(B), shifts, w.tol, w.max_iter)
    p = ms.msolve_cgm(A, dev(w.b), shifts, w.tol, w.max_iter)
    assert g.iterations == p.iterations and torch.equal(g.x, p.x)
    # one system
    g = ms.msolve_solve_multirhs(A, ms.MSOLVE_ALG_CGM, dev(w.b[None, :]), [0.3], w.tol, w.max_iter)
    p = ms.msolve_cgm(A, dev(w.b), [0.3], w.tol, w.max_iter)
    assert torch.equal(g.x, p.x)
    with pytest.raises(ms.MsolveError):
        ms.msolve_solve_multirhs(A, ms.MSOLVE_ALG_CGM, dev(B[:2]), [0.5, 0.5], 1e-10, 10)
    # the handle still serves ordinary solves afterwards (thresholds back to ||b||)
    p2 = ms.msolve_cgm(A, dev(w.b), shifts, w.tol, w.max_iter)
    o = oracle.cgm(w.rowptr, w.colidx, w.val, w.b, shifts, w.tol, w.max_iter)
    assert p2.iterations == o.iterations and np.array_equal(p2.conv_iter, o.conv_iter)
    ms.msolve_destroy(A)
