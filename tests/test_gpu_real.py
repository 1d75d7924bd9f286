"""GPU parity for the REAL element types (MSOLVE_F32 / MSOLVE_F64): the paper's own workload,
2-D 5-point Poisson with 15 shifts (Table 1), plus a real
non-symmetric convection-diffusion matrix for BiCGStab-M.  Same bars as the complex types:
relative L2 difference to the oracle <= 1e-9 (float64) / 1e-4 (float32), true residual <= 10 tol,
iteration counts within +-2."""
import numpy as np
import pytest
import scipy.sparse as sp
import torch

import oracle
from paper_1102_2143_b200 import workloads as W

pytestmark = pytest.mark.gpu

REL = {np.float64: 1e-9, np.float32: 1e-4}
TOL = {np.float64: 1e-10, np.float32: 1e-5}


@pytest.fixture(scope="module")
def ms():
    from paper_1102_2143_b200 import binding, build
    build.build()
    binding.load_library()
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def solve_both(ms, w, dtype, flags, tol):
    A = ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val.astype(dtype)), flags)
    if flags == 1:      # VECTOR by name: through the graph of kernels (AUTO, flags = 0, takes the one-kernel path at these sizes)
        ms.msolve_config(A, ms.MSOLVE_CFG_ITER_PATH, 1)
    fn, ofn = (ms.msolve_cgm, oracle.cgm) if w.algorithm == "cgm" else (ms.msolve_bicgstabm, oracle.bicgstabm)
    g = fn(A, dev(w.b.astype(dtype)), w.shifts, tol, w.max_iter)
    x = g.x.cpu().numpy()
    ms.msolve_destroy(A)
    o = ofn(w.rowptr, w.colidx, w.val.astype(dtype), w.b.astype(dtype), w.shifts, tol, w.max_iter)
    assert x.dtype == dtype and o.x.dtype == dtype
    assert g.status == o.status == oracle.OK
    assert abs(g.iterations - o.iterations) <= 2
    assert np.all(np.abs(g.conv_iter - o.conv_iter) <= 2)
    M = sp.csr_matrix((w.val, w.colidx, w.rowptr), shape=(w.n, w.n))
    for k, s in enumerate(w.shifts):
        xk = x[k].astype(np.float64)
        d = np.linalg.norm(xk - o.x[k].astype(np.float64)) / np.linalg.norm(o.x[k])
        assert d <= REL[dtype], (k, d)
        true = np.linalg.norm(w.b - (M @ xk + s * xk)) / np.linalg.norm(w.b)
        assert true <= 10.0 * tol, (k, true)
    return g, o


@pytest.mark.parametrize("flags", [0, 1, 2, 3])                   # AUTO, VECTOR, MERGE, TILE
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_spmv_real(ms, dtype, flags):
    w = W.poisson_workload(67, 45, real=True)                     # n = 3015: odd, ragged tiles
    A = ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val.astype(dtype)), flags)
    x = np.random.default_rng(3).standard_normal(w.n).astype(dtype)
    y, dot = ms.msolve_spmv(A, dev(x))
    ref = oracle.spmv(w.rowptr, w.colidx, w.val.astype(dtype), x)
    eps = np.finfo(dtype).eps
    assert np.max(np.abs(y.cpu().numpy() - ref)) <= 16 * eps * np.max(np.abs(ref))
    assert abs(dot - np.dot(x.astype(np.float64), ref.astype(np.float64))) <= 1e-6 * abs(dot) and dot.imag == 0.0
    ms.msolve_destroy(A)


@pytest.mark.parametrize("flags", [0, 1, 2, 3])
@pytest.mark.parametrize("dtype,shape", [(np.float64, (64, 48)), (np.float64, (37, 29)), (np.float32, (24, 20)),
                                         (np.float32, (23, 19))])
def test_poisson_cgm_real(ms, dtype, shape, flags):
    # 15 shifts as in Table 1; odd sizes exercise the scalar (non-16-byte) element-wise path
    w = W.poisson_workload(shape[0], shape[1], nshifts=15, real=True)
    g, o = solve_both(ms, w, dtype, flags, TOL[dtype])
    assert np.all(np.diff(g.conv_iter) <= 0)


@pytest.mark.parametrize("dtype,shape", [(np.float64, (40, 36)), (np.float32, (21, 18))])
def test_convection_diffusion_bicgstabm_real(ms, dtype, shape):
    w = W.poisson_workload(shape[0], shape[1], nshifts=8, real=True, drift=0.4)
    assert w.algorithm == "bicgstabm"
    solve_both(ms, w, dtype, 0, TOL[dtype] * 10)


def test_real_matches_complex_embedding_on_gpu(ms):
    # the same real problem through the complex128 kernels gives the same solutions (rounding level)
    w = W.poisson_workload(32, 32, nshifts=5, real=True)
    A = ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val))
    Ac = ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val.astype(np.complex128)))
    g = ms.msolve_cgm(A, dev(w.b), w.shifts, 1e-10, w.max_iter)
    gc = ms.msolve_cgm(Ac, dev(w.b.astype(np.complex128)), w.shifts, 1e-10, w.max_iter)
    assert g.iterations == gc.iterations
    xc = gc.x.cpu().numpy()
    assert np.abs(xc.imag).max() == 0.0
    assert np.allclose(g.x.cpu().numpy(), xc.real, rtol=0, atol=1e-13 * np.abs(xc).max())
    ms.msolve_destroy(A); ms.msolve_destroy(Ac)


def test_bsr3_rejects_real(ms):
    w = W.config2(extents=(4, 4, 4, 4))
    with pytest.raises(ms.MsolveError):
        ms.msolve_create_bsr3(dev(w.browptr), dev(w.bcolidx), dev(w.blocks.real.copy()))
