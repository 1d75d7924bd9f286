"""Host-side pin of the algebra behind MSOLVE_CFG_DEFER_UPDATE ("Deferred multishift update").

No GPU and no library code: a plain numpy CG-M in the lagged form the kernels use (p_k(n) = zeta_k(n) r_n +
alpha_k(n) p_k(n-1), x_k(n+1) = x_k(n) - beta_k(n) p_k(n)) is run once step by step and once with the per-chunk
coefficient recurrences the scalar kernel keeps (Cp, Cx, Ap, Ax), flushing every M iterations; both must give the
same x_k and p_k to rounding, for every chunk length, and both must solve the shifted systems (dense LU).
The recurrences for zeta, alpha, beta are Alg. 1 l.20-26 as the oracle reads them."""
import numpy as np
import pytest


def _cgm_scalars_and_residuals(A, b, shifts, iters):
    """Step-by-step CG-M on the base system; returns per iteration (r_n, zeta_k(n), alpha_k(n), beta_k(n))."""
    S = len(shifts)
    r, p = b.copy(), b.copy()
    zeta_prev, zeta = np.ones(S), np.ones(S)
    alpha, beta_prev = 0.0, 1.0
    alpha_k = np.zeros(S)
    R0 = np.vdot(r, r).real
    out = []
    for n in range(iters):
        if n > 0:
            p = r + alpha * p
        q = A @ p
        beta = -R0 / np.vdot(p, q).real
        zeta_new = zeta * zeta_prev * beta_prev / (beta * alpha * (zeta_prev - zeta) + zeta_prev * beta_prev * (1.0 - shifts * beta))
        beta_k = beta * zeta_new / zeta
        out.append((r.copy(), zeta.copy(), alpha_k.copy(), beta_k.copy()))
        r = r + beta * q
        R1 = np.vdot(r, r).real
        alpha = R1 / R0
        alpha_k = alpha * (zeta_new / zeta) ** 2
        zeta_prev, zeta, beta_prev, R0 = zeta, zeta_new, beta, R1
    return out


def _stepwise(steps, n, S):
    x = np.zeros((S, n), dtype=complex)
    p = np.zeros((S, n), dtype=complex)
    for it, (r, z, ak, bk) in enumerate(steps):
        p = r[None, :] if it == 0 else z[:, None] * r[None, :] + ak[:, None] * p
        x = x - bk[:, None] * p
    return x, p


def _deferred(steps, n, S, M):
    x = np.zeros((S, n), dtype=complex)            # X_k, P_k "in memory"
    p = np.zeros((S, n), dtype=complex)
    chunk, Cp, Cx, Ap, Ax = [], np.zeros((S, M)), np.zeros((S, M)), np.ones(S), np.zeros(S)

    def flush():
        nonlocal x, p, chunk, Cp, Cx, Ap, Ax
        R = np.array(chunk)                        # [f, n]
        f = len(chunk)
        x = x + Ax[:, None] * p + Cx[:, :f] @ R
        p = Ap[:, None] * p + Cp[:, :f] @ R
        chunk, Cp, Cx, Ap, Ax = [], np.zeros((S, M)), np.zeros((S, M)), np.ones(S), np.zeros(S)

    for it, (r, z, ak, bk) in enumerate(steps):
        f = len(chunk)
        if it == 0:
            ak = np.zeros(S)                       # p_k(0) = r_0: zeta = 1 and nothing carried over
        Cp[:, :f] *= ak[:, None]
        Cp[:, f] = z
        Ap = ak * Ap
        Cx[:, :f + 1] -= bk[:, None] * Cp[:, :f + 1]
        Ax = Ax - bk * Ap
        chunk.append(r)
        if len(chunk) == M:
            flush()
    if chunk:
        flush()
    return x, p


@pytest.mark.parametrize("M", [1, 2, 3, 5, 8, 32])
def test_chunked_coefficients_reproduce_the_stepwise_update(M):
    rng = np.random.default_rng(7)
    n, S, iters = 40, 5, 17
    G = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    A = G @ G.conj().T / n + 0.5 * np.eye(n)       # Hermitian positive definite
    b = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    b /= np.linalg.norm(b)
    shifts = np.array([0.0, 0.05, 0.3, 1.0, 4.0])
    steps = _cgm_scalars_and_residuals(A, b, shifts, iters)
    xs, ps = _stepwise(steps, n, S)
    xd, pd = _deferred(steps, n, S, M)
    assert np.allclose(xd, xs, rtol=0, atol=1e-13 * np.abs(xs).max())
    assert np.allclose(pd, ps, rtol=0, atol=1e-13 * max(np.abs(ps).max(), 1e-300))
    # and the iterates are what the method promises: after enough iterations x_k solves (A + sigma_k) x = b
    steps = _cgm_scalars_and_residuals(A, b, shifts, 60)
    xd, _ = _deferred(steps, n, S, M)
    for k, s in enumerate(shifts):
        ref = np.linalg.solve(A + s * np.eye(n), b)
        assert np.linalg.norm(xd[k] - ref) <= 1e-10 * np.linalg.norm(ref), (M, k)
