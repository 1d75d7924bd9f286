"""GPU parity of the matrix-free SU(3) lattice operator (msolve_create_lattice_su3; SURVEY.md
8(f)-2) against the CPU oracle run on the ASSEMBLED matrix of the same links."""
import numpy as np
import pytest

import oracle
from paper_1102_2143_b200 import workloads as W
import test_gpu_parity
from test_gpu_parity import check_parity, dev, gpu_solve, make_matrix, ms, oracle_solve  # noqa: F401

pytestmark = pytest.mark.gpu


def _workload(extents, nonhermitian=False):
    d = len(extents)
    if nonhermitian:
        return W.su3_workload("lat_nh", "bicgstabm", extents, d + 0.2, 0.6, 0.4, np.array([0.0, 0.1, 1.0]), 1e-9)
    return W.su3_workload("lat_h", "cgm", extents, 0.05 ** 2 + 2 * d, 1.0, 1.0, W.log_shifts(1e-3, 1.0, 5), 1e-10)


EXTENTS = [(4, 4, 6, 5),        # 8 x0-rows per tile
           (12, 10, 9, 11),     # 2 rows per tile, odd row count: ragged last tile, many tiles per CTA
           (32, 4, 3, 3),       # one row per tile (the config-4 shape); blocked kernel: complex128 only (2 x 1 block)
           (32, 6, 4, 3),       # blocked kernel in both precisions: 3 x 2 blocks per x3-slice, several tiles per stage
           (32, 4, 4, 3),       # blocked kernel, two blocks per direction: both neighbours of a block are the same block
           (5, 3, 4),           # 3-D, odd L0: complex64 rows are not 16-byte multiples -> row kernel
           (3, 3),              # 2-D, smallest legal extents
           (16,),               # 1-D
           (36, 3, 3, 3)]       # L0 > 32 sites: row kernel


@pytest.fixture(params=[1, 2, 3, 4], ids=["termsite", "warptile", "hybrid", "blocked"])
def tile_kernel(request, ms):
    """Run with each of the tile kernels forced (default: the faster one per element type; the blocked kernel
    leaves lattices it does not cover -- L0 != 32, fewer than 4 dimensions, odd extents -- to the default)."""
    test_gpu_parity.FORCED_CFG[ms.MSOLVE_CFG_LATTICE_KERNEL] = request.param
    yield request.param
    test_gpu_parity.FORCED_CFG.clear()


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("fmt", ["lat", "latrows"])
@pytest.mark.parametrize("nh", [False, True])
@pytest.mark.parametrize("extents", EXTENTS)
def test_lattice_spmv_matches_oracle(ms, tile_kernel, extents, nh, fmt, dtype):
    w = _workload(extents, nh)
    rng = np.random.default_rng(5)
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


@pytest.mark.parametrize("fmt", ["lat", "latrows"])
@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
def test_config2_cgm_matrix_free(ms, fmt, dtype, tol):
    w = W.config2()
    g = gpu_solve(ms, w, dtype, fmt, tol=tol)
    o = oracle_solve(w, dtype, tol=tol)
    check_parity(w, dtype, g, o, tol)


@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 1e-5)])
def test_config4_scaled_cgm_matrix_free(ms, tile_kernel, dtype, tol):
    w = W.config4(extents=(32, 8, 4, 6), tol=tol)
    g = gpu_solve(ms, w, dtype, "lat")
    o = oracle_solve(w, dtype)
    check_parity(w, dtype, g, o, tol)


def test_blocked_kernel_is_bit_identical_to_the_warp_kernel(ms):
    # same operands, same order of multiply-adds per site: only where the operands come from differs
    for nh in (False, True):
        w = _workload((32, 6, 4, 3), nh)
        rng = np.random.default_rng(7)
        for dtype in (np.complex128, np.complex64):
            x = (rng.standard_normal(w.n) + 1j * rng.standard_normal(w.n)).astype(dtype)
            ys = []
            for kern in (2, 4):
                A = make_matrix(ms, w, dtype, "lat", cfg={ms.MSOLVE_CFG_LATTICE_KERNEL: kern})
                y, _ = ms.msolve_spmv(A, dev(x))
                ys.append(y.cpu().numpy())
                ms.msolve_destroy(A)
            assert np.array_equal(ys[0], ys[1])


@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-9), (np.complex64, 1e-4)])
def test_bicgstabm_on_the_blocked_kernel(ms, dtype, tol):
    # both BiCGStab-M SpMV roles (two and five fused dot products) on a lattice the blocked kernel covers
    w = W.config3(extents=(32, 4, 4, 3))
    w.tol = tol
    g = gpu_solve(ms, w, dtype, "lat", cfg={ms.MSOLVE_CFG_LATTICE_KERNEL: 4})
    o = oracle_solve(w, dtype)
    check_parity(w, dtype, g, o, tol)


@pytest.mark.parametrize("fmt", ["lat", "latrows"])
def test_config3_bicgstabm_matrix_free(ms, tile_kernel, fmt):
    w = W.config3(extents=(8, 8, 8, 8))
    g = gpu_solve(ms, w, np.complex128, fmt)
    o = oracle_solve(w, np.complex128)
    check_parity(w, np.complex128, g, o, w.tol)


def test_lattice_create_validation(ms):
    import torch
    links = torch.zeros(4 * 81 * 9, dtype=torch.complex128, device="cuda")
    with pytest.raises(ms.MsolveError):
        ms.msolve_create_lattice_su3((3, 3, 3, 3, 1), torch.zeros(5 * 81 * 9, dtype=torch.complex128, device="cuda"), 8.0, 1.0, 1.0)
    with pytest.raises(ms.MsolveError):
        ms.msolve_create_lattice_su3((3, 3, 3, 3), links, float("nan"), 1.0, 1.0)
    with pytest.raises(ms.MsolveError):
        ms.msolve_create_lattice_su3((3, 3, 3, 3), links.real.contiguous(), 8.0, 1.0, 1.0)
    with pytest.raises(ValueError):
        ms.msolve_create_lattice_su3((3, 3, 3), links, 8.0, 1.0, 1.0)
