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


def _rhs(seed, s, n, dtype, smooth):
    rng = np.random.default_rng(seed)
    if smooth is None:                      # independent Gaussian right-hand sides of different norms
        B = rng.standard_normal((s, n)) + 1j * rng.standard_normal((s, n))
        B /= np.linalg.norm(B, axis=1)[:, None]
        B *= np.linspace(1.0, 3.0, s)[:, None]
    else:                                   # b_i = c_0 + sigma_i c_1 + sigma_i^2 c_2: smooth in the shift
        c = rng.standard_normal((3, n)) + 1j * rng.standard_normal((3, n))
        B = np.array([c[0] + t * c[1] + t * t * c[2] for t in smooth])
        B /= np.linalg.norm(B[0])
    return B.astype(dtype)


@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
@pytest.mark.parametrize("alg,fmt", [("cgm", "bsr3"), ("cgm", "csr"), ("bicgstabm", "bsr3"), ("cgm", "lat")])
def test_multirhs_matches_oracle(ms, alg, fmt, dtype, tol):
    w = W.config2(extents=(6, 6, 4, 6)) if alg == "cgm" else W.config3(extents=(6, 6, 4, 6))
    code = ms.MSOLVE_ALG_CGM if alg == "cgm" else ms.MSOLVE_ALG_BICGSTABM
    shifts = np.array([0.0, 0.4, 1.0, 1.7, 2.5])
    B = _rhs(31, shifts.size, w.n, dtype, None)
    A = make_matrix(ms, w, dtype, fmt)
    g = ms.msolve_solve_multirhs(A, code, dev(B), shifts, tol, w.max_iter)
    o = oracle.multirhs(w.rowptr, w.colidx, w.val.astype(dtype), B, shifts, tol, w.max_iter, alg)
    assert g.status == o.status == 0 and abs(g.iterations - o.iterations) <= 2
    assert np.all(np.abs(g.conv_iter - o.conv_iter) <= 2)
    M = sp.csr_matrix((w.val, w.colidx, w.rowptr), shape=(w.n, w.n))
    x = g.x.cpu().numpy()
    for i, s in enumerate(shifts):
        diff = x[i].astype(np.complex128) - o.x[i]
        assert np.linalg.norm(diff) <= REL[dtype] * np.linalg.norm(o.x[i]), (i, np.linalg.norm(diff) / np.linalg.norm(o.x[i]))
        assert np.abs(diff).max() <= MAXABS_C * REL[dtype] * np.abs(o.x[i]).max(), i
        xi = x[i].astype(np.complex128)
        bi = B[i].astype(np.complex128)
        assert np.linalg.norm(bi - (M @ xi + s * xi)) <= 10 * tol * np.linalg.norm(bi), i     # relative to ITS rhs
        assert g.relres[i] <= tol * (1 + 1e-9)
    ms.msolve_destroy(A)


def test_multirhs_many_shifts_smooth_rhs(ms):
    # 20 shifts (> 16: the level-by-level divided-difference path and the generic guess kernel), right-hand sides
    # smooth in the shift, so the divided differences beyond the third vanish up to rounding
    w = W.config2(extents=(4, 6, 4, 6))
    shifts = np.linspace(0.05, 2.0, 20)
    B = _rhs(32, 20, w.n, np.complex128, shifts)
    A = make_matrix(ms, w, np.complex128, "bsr3")
    g = ms.msolve_solve_multirhs(A, ms.MSOLVE_ALG_CGM, dev(B), shifts, 1e-10, w.max_iter)
    o = oracle.multirhs(w.rowptr, w.colidx, w.val, B, shifts, 1e-10, w.max_iter)
    assert g.status == o.status == 0 and abs(g.iterations - o.iterations) <= 2
    x = g.x.cpu().numpy()
    M = sp.csr_matrix((w.val, w.colidx, w.rowptr), shape=(w.n, w.n))
    for i, s in enumerate(shifts):
        # the construction itself loses digits here (weights up to prod |sigma_i - sigma_j|): GPU and oracle agree to
        # what the arithmetic allows, and both solve the systems
        assert np.linalg.norm(x[i] - o.x[i]) <= 1e-7 * np.linalg.norm(o.x[i]), i
        assert np.linalg.norm(B[i] - (M @ x[i] + s * x[i])) <= 1e-6 * np.linalg.norm(B[i]), i
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
