"""The whole solve as ONE cooperative kernel (MSOLVE_CFG_ITER_PATH = 2, csrc/fused_small.cu): the path AUTO takes for
systems that live in L2 (BASELINE configs 1 and 2).  Same bars against the oracle as the graph path, agreement with
the graph path to rounding, and the same edge cases."""
import numpy as np
import pytest
import torch

import oracle
from paper_1102_2143_b200 import workloads as W
from test_gpu_parity import HIST_RTOL, HIST_ULPS, REL, check_parity, dev, gpu_solve, make_matrix, ms, oracle_solve  # noqa: F401

pytestmark = pytest.mark.gpu


def fused(ms):
    return {ms.MSOLVE_CFG_ITER_PATH: 2}


def resident(ms):
    return {ms.MSOLVE_CFG_ITER_PATH: 3}


@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
@pytest.mark.parametrize("which,fmt", [("c1", "csr"), ("c2", "csr"), ("c2", "bsr3"), ("c2", "csrtile"), ("c5", "csrvector"), ("c2odd", "bsr3"),
                                       ("c4s", "bsr3"), ("c3s", "bsr3"), ("c3s", "csr")])
def test_resident_matches_oracle_and_graph(ms, which, fmt, dtype, tol):
    # MSOLVE_CFG_ITER_PATH = 3 (csrc/resident.cu): matrix and all vectors in shared memory for the whole solve
    w = {"c1": W.config1, "c2": W.config2, "c2odd": lambda: W.config2(extents=(5, 3, 7, 3)),
         "c5": lambda: W.config5(n=(1 << 13) + 13), "c4s": lambda: W.config4(extents=(8, 8, 8, 16), want_csr=True),
         "c3s": lambda: W.config3(extents=(8, 8, 6, 6))}[which]()          # BiCGStab-M
    w.tol = 10 * tol if which == "c3s" else tol
    g = gpu_solve(ms, w, dtype, fmt, cfg=resident(ms))
    o = oracle_solve(w, dtype)
    check_parity(w, dtype, g, o, w.tol)
    assert g[5] == 1
    gg = gpu_solve(ms, w, dtype, fmt)
    assert abs(gg[1] - g[1]) <= 1
    for k in range(w.shifts.size):
        d = np.linalg.norm(g[2][k].astype(np.complex128) - gg[2][k]) / np.linalg.norm(gg[2][k])
        assert d <= REL[dtype], (k, d)
    g2 = gpu_solve(ms, w, dtype, fmt, cfg=resident(ms))
    assert g2[1] == g[1] and np.array_equal(g2[2], g[2]) and np.array_equal(g2[3], g[3])


@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
@pytest.mark.parametrize("which,fmt", [("c1", "csr"), ("c2", "csr"), ("c2", "bsr3"), ("c2", "bsr3rows"), ("c2", "lat"), ("c2", "latrows"),
                                       ("c5", "csrvector"), ("c3", "csr"), ("c3", "bsr3"), ("c3", "lat"), ("c2odd", "bsr3")])
def test_fused_matches_oracle_and_graph(ms, which, fmt, dtype, tol):
    w = {"c1": W.config1, "c2": W.config2, "c2odd": lambda: W.config2(extents=(5, 3, 7, 3)),
         "c5": lambda: W.config5(n=(1 << 14) + 13), "c3": lambda: W.config3(extents=(8, 8, 8, 8))}[which]()
    w.tol = 10 * tol if which == "c3" else tol
    g = gpu_solve(ms, w, dtype, fmt, cfg=fused(ms))
    o = oracle_solve(w, dtype)
    check_parity(w, dtype, g, o, w.tol)
    assert g[5] == 1                                        # ONE kernel launch for init + every iteration
    gg = gpu_solve(ms, w, dtype, fmt)                       # the graph of kernels on the same inputs
    assert abs(gg[1] - g[1]) <= 1
    for k in range(w.shifts.size):
        d = np.linalg.norm(g[2][k].astype(np.complex128) - gg[2][k]) / np.linalg.norm(gg[2][k])
        assert d <= REL[dtype], (k, d)          # two groupings of the same dot products: rounding, amplified by the iteration
    # bit-reproducible: the same solve again returns the same bytes
    g2 = gpu_solve(ms, w, dtype, fmt, cfg=fused(ms))
    assert g2[1] == g[1] and np.array_equal(g2[2], g[2]) and np.array_equal(g2[3], g[3])


@pytest.mark.parametrize("which,fmt", [("c2", "bsr3"), ("c3", "lat")])
def test_phase_clock_counts_iterations_and_changes_nothing(ms, which, fmt):
    # msolve_set_phase_clock: slot 15 counts the iterations of every solve, the phase slots of the algorithm are all
    # non-zero, the rest stay zero, and the solve returns the same bytes with the clock on and off
    w = W.config2() if which == "c2" else W.config3(extents=(8, 8, 8, 8))
    g = gpu_solve(ms, w, np.complex128, fmt, cfg=fused(ms))
    A = make_matrix(ms, w, np.complex128, fmt, cfg=fused(ms))
    ns = torch.zeros(16, dtype=torch.int64, device="cuda")
    ms.msolve_set_phase_clock(A, ns)
    solve = ms.msolve_cgm if w.algorithm == "cgm" else ms.msolve_bicgstabm
    b = dev(w.b)
    for _ in range(2):
        res = solve(A, b, w.shifts, w.tol, w.max_iter)
    t = ns.cpu().numpy()
    nph = 6 if w.algorithm == "cgm" else 8
    assert t[15] == 2 * res.iterations == 2 * g[1]
    assert np.all(t[:nph] > 0) and np.all(t[nph:15] == 0)
    assert t[:nph].sum() < 1e9                              # two small solves: well under a second
    assert np.array_equal(res.x.cpu().numpy(), g[2])
    ms.msolve_set_phase_clock(A, None)
    solve(A, b, w.shifts, w.tol, w.max_iter)
    assert ns.cpu().numpy()[15] == t[15]
    ms.msolve_destroy(A)


def test_resident_needs_the_problem_to_fit(ms):
    # 16 shifts x 49152 rows x 16 B: 35 vectors + matrix = 49 MB do not fit in 148 x 200 KB; asking for the path by
    # name is an error, AUTO falls back to the L2 one-kernel path
    w = W.config4(extents=(8, 8, 16, 16))
    A = ms.msolve_create_bsr3(dev(w.browptr), dev(w.bcolidx), dev(w.blocks))
    ms.msolve_config(A, ms.MSOLVE_CFG_ITER_PATH, 3)
    with pytest.raises(ms.MsolveError):
        ms.msolve_cgm(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    ms.msolve_config(A, ms.MSOLVE_CFG_ITER_PATH, 0)
    r = ms.msolve_cgm(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    assert r.status == 0 and ms.msolve_last_launch_count(A) == 1
    ms.msolve_destroy(A)


def test_auto_picks_by_footprint(ms):
    # AUTO (the library default): one kernel for config 2 (11 MB: resident in shared memory; BiCGStab-M: the L2 path),
    # the graph of kernels for a system beyond the 256 MB bound
    w = W.config2()
    A = ms.msolve_create_bsr3(dev(w.browptr), dev(w.bcolidx), dev(w.blocks))
    r = ms.msolve_cgm(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    assert r.status == 0 and ms.msolve_last_launch_count(A) == 1
    ms.msolve_config(A, ms.MSOLVE_CFG_ITER_PATH, 1)
    r1 = ms.msolve_cgm(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    assert ms.msolve_last_launch_count(A) == 2 + 6 * r1.iterations      # the sixth kernel: the flush of the deferred update
    ms.msolve_destroy(A)
    w = W.config4(extents=(16, 16, 16, 32))                # 393216 rows, 16 shifts: 36 vectors of 6.3 MB + 175 MB of matrix
    A = ms.msolve_create_bsr3(dev(w.browptr), dev(w.bcolidx), dev(w.blocks))
    r = ms.msolve_cgm(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    assert r.status == 0 and ms.msolve_last_launch_count(A) == 2 + 6 * r.iterations
    ms.msolve_destroy(A)
    # kernels the L2 one-kernel path does not cover stay on the graph path (here a system too large for shared
    # memory); asking for the one-kernel path by name is an error
    w = W.config4(extents=(8, 8, 8, 16), want_csr=True)
    A = ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val), ms.MSOLVE_SPMV_MERGE)
    r = ms.msolve_cgm(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    assert ms.msolve_last_launch_count(A) == 2 + 7 * r.iterations      # merge-path SpMV = two launches
    ms.msolve_config(A, ms.MSOLVE_CFG_ITER_PATH, 2)
    with pytest.raises(ms.MsolveError):
        ms.msolve_cgm(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    ms.msolve_destroy(A)


@pytest.mark.parametrize("alg,path", [("cgm", 2), ("bicgstabm", 2), ("cgm", 3), ("bicgstabm", 3)])
def test_fused_edge_cases(ms, alg, path):
    w = W.config2(extents=(4, 4, 4, 4)) if alg == "cgm" else W.config3(extents=(4, 4, 4, 4))
    fn = ms.msolve_cgm if alg == "cgm" else ms.msolve_bicgstabm
    A = make_matrix(ms, w, np.complex128, "bsr3", cfg={ms.MSOLVE_CFG_ITER_PATH: path})
    S = w.shifts.size
    x = torch.full((S, w.n), 7.0, dtype=torch.complex128, device="cuda")
    r = fn(A, torch.zeros(w.n, dtype=torch.complex128, device="cuda"), w.shifts, 1e-10, 100, x=x)       # b = 0
    assert r.status == ms.MSOLVE_OK and r.iterations == 0 and not r.x.abs().max().item() and np.all(r.conv_iter == 0)
    x.fill_(7.0)
    r = fn(A, dev(w.b), w.shifts, 1e-10, 0, x=x)                                                         # max_iter = 0
    assert r.status == ms.MSOLVE_MAXITER and r.iterations == 0 and not r.x.abs().max().item()
    for nit in (1, 2, 5):                                                                                # stopped early
        r = fn(A, dev(w.b), w.shifts, 0.0, nit)
        o = oracle_solve(w, np.complex128, tol=0.0, max_iter=nit)
        assert r.status == o.status == oracle.MAXITER and r.iterations == nit
        xg = r.x.cpu().numpy()
        for k in range(S):
            assert np.linalg.norm(xg[k] - o.x[k]) / np.linalg.norm(o.x[k]) < 1e-12
        assert np.allclose(r.relres, o.relres, rtol=1e-10)
    # stop rule 1 and the scalar history through the one-kernel path
    ms.msolve_config(A, ms.MSOLVE_CFG_STOP_RULE, 1)
    cols = 3 + 3 * S if alg == "cgm" else 8 + 6 * S
    hist = torch.zeros((64, cols), dtype=torch.float64, device="cuda")
    ms.msolve_set_history(A, hist)
    r = fn(A, dev(w.b), w.shifts, w.tol, w.max_iter)
    ofn = oracle.cgm if alg == "cgm" else oracle.bicgstabm
    o = ofn(w.rowptr, w.colidx, w.val, w.b, w.shifts, w.tol, w.max_iter, stop_rule=1, hist_cap=64)
    assert r.status == o.status == 0 and r.iterations == o.iterations and np.all(r.conv_iter == o.iterations)
    hg = hist.cpu().numpy()[: o.iterations]
    rr = o.hist[:, 2] if alg == "cgm" else o.hist[:, 6]
    bar = HIST_RTOL + HIST_ULPS * np.finfo(np.float64).eps * (np.arange(o.iterations) + 1) / np.sqrt(rr)
    keep = np.abs(o.hist) > 0
    dev_rel = np.where(keep, np.abs(hg - o.hist) / np.where(keep, np.abs(o.hist), 1.0), 0.0)
    if alg == "bicgstabm":          # components of complex scalars: relative to the modulus of the pair
        zg = np.delete(hg, [6, 7], axis=1).copy().view(np.complex128)
        zo = np.delete(o.hist, [6, 7], axis=1).copy().view(np.complex128)
        dev_rel = np.abs(zg - zo) / np.abs(zo)
    assert np.all(dev_rel.max(axis=1) <= bar), (dev_rel.max(axis=1) / bar).max()
    ms.msolve_destroy(A)


@pytest.mark.parametrize("path", [2, 3])
def test_fused_multirhs_and_real(ms, path):
    w = W.config2(extents=(4, 6, 4, 6))
    shifts = np.array([0.0, 0.4, 1.0, 1.7])
    rng = np.random.default_rng(41)
    B = rng.standard_normal((4, w.n)) + 1j * rng.standard_normal((4, w.n))
    B = B[0] + shifts[:, None] * B[1] + 0.05 * B
    A = make_matrix(ms, w, np.complex128, "bsr3", cfg={ms.MSOLVE_CFG_ITER_PATH: path})
    g = ms.msolve_solve_multirhs(A, ms.MSOLVE_ALG_CGM, dev(B), shifts, 1e-10, w.max_iter)
    o = oracle.multirhs(w.rowptr, w.colidx, w.val, B, shifts, 1e-10, w.max_iter)
    assert g.status == o.status == 0 and abs(g.iterations - o.iterations) <= 2
    x = g.x.cpu().numpy()
    for i in range(4):
        assert np.linalg.norm(x[i] - o.x[i]) <= 1e-9 * np.linalg.norm(o.x[i])
    ms.msolve_destroy(A)
    # real element types (the paper's own workload shape), odd size: scalar element-wise path
    w = W.poisson_workload(37, 29, nshifts=15, real=True)
    for dtype, tol, bar in ((np.float64, 1e-10, 1e-9), (np.float32, 1e-5, 1e-4)):
        A = ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val.astype(dtype)), ms.MSOLVE_SPMV_VECTOR)
        ms.msolve_config(A, ms.MSOLVE_CFG_ITER_PATH, path)
        g = ms.msolve_cgm(A, dev(w.b.astype(dtype)), w.shifts, tol, w.max_iter)
        o = oracle.cgm(w.rowptr, w.colidx, w.val.astype(dtype), w.b.astype(dtype), w.shifts, tol, w.max_iter)
        assert g.status == o.status == 0 and abs(g.iterations - o.iterations) <= 2 and ms.msolve_last_launch_count(A) == 1
        x = g.x.cpu().numpy()
        for k in range(15):
            assert np.linalg.norm(x[k].astype(np.float64) - o.x[k]) <= bar * np.linalg.norm(o.x[k])
        ms.msolve_destroy(A)
