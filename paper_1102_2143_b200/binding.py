"""Thin Python binding of the C ABI in include/msolve.h (argument marshalling only).

Same names as the C entry points.  PyTorch is used for device memory and streams; every step
of the solver path runs inside libmsolve.so's CUDA kernels.  There is NO fallback: if the
library is missing or fails to load, every call raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmsolve.so")

MSOLVE_C64, MSOLVE_C128, MSOLVE_F32, MSOLVE_F64 = 0, 1, 2, 3
MSOLVE_ALG_CGM, MSOLVE_ALG_BICGSTABM = 0, 1
MSOLVE_OK, MSOLVE_MAXITER, MSOLVE_BREAKDOWN = 0, 1, 2
MSOLVE_EINVAL, MSOLVE_ECUDA, MSOLVE_ENOMEM = -1, -2, -3
MSOLVE_SPMV_AUTO, MSOLVE_SPMV_VECTOR, MSOLVE_SPMV_MERGE, MSOLVE_SPMV_TILE = 0, 1, 2, 3
MSOLVE_MAX_SHIFTS = 128
MSOLVE_CFG_LOOP_MODE = 0
MSOLVE_CFG_UPDATE_KERNEL = 1
MSOLVE_CFG_LATTICE_KERNEL = 2
MSOLVE_CFG_STOP_RULE = 3
MSOLVE_CFG_X_WINDOW = 4
MSOLVE_CFG_MATRIX_L2 = 5
MSOLVE_CFG_ITER_PATH = 6
MSOLVE_CFG_FUSED_CTAS = 7
MSOLVE_CFG_MATRIX_L2_KEEP_PERCENT = 8
MSOLVE_CFG_DEFER_UPDATE = 9

EXPORTS = (
    "msolve_create_csr", "msolve_create_bsr3", "msolve_create_lattice_su3", "msolve_workspace_bytes", "msolve_cgm",
    "msolve_bicgstabm", "msolve_multirhs_workspace_bytes", "msolve_solve_multirhs", "msolve_solve_host", "msolve_solve_host_batch", "msolve_spmv", "msolve_spmv_csr_noalloc", "msolve_profile_iteration",
    "msolve_kernel_name", "msolve_last_launch_count", "msolve_config", "msolve_set_history", "msolve_set_phase_clock", "msolve_destroy",
    "msolve_last_error",
    "msolve_slab_plan_create", "msolve_slab_plan_nlocal", "msolve_slab_plan_nhalo", "msolve_slab_plan_npeers",
    "msolve_slab_plan_peer", "msolve_slab_plan_colidx", "msolve_slab_plan_destroy",
    "msolve_slabs_create_csr", "msolve_slabs_create_bsr3", "msolve_slabs_count", "msolve_slabs_halo_elements",
    "msolve_slabs_workspace_bytes", "msolve_slabs_cgm", "msolve_slabs_bicgstabm", "msolve_slabs_spmv",
    "msolve_slabs_last_launch_count", "msolve_slabs_destroy",
)

_lib = None


class MsolveError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__("msolve error %d: %s" % (code, text))
        self.code = code


def load_library() -> ctypes.CDLL:
    """dlopen libmsolve.so and declare the prototypes.  Raises if it is not there."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("libmsolve.so is not built (run `python -m paper_1102_2143_b200.build` "
                           "or __graft_entry__.build()); there is no CPU fallback")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, dbl, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_double, ctypes.c_size_t
    lib.msolve_create_csr.argtypes = [ctypes.POINTER(vp), i64, i64, vp, vp, vp, i32, i32, vp]
    lib.msolve_create_bsr3.argtypes = [ctypes.POINTER(vp), i64, i64, vp, vp, vp, i32, i32, vp]
    lib.msolve_create_lattice_su3.argtypes = [ctypes.POINTER(vp), i32, vp, vp, dbl, dbl, dbl, i32, i32, vp]
    lib.msolve_workspace_bytes.argtypes = [vp, i32, i32]
    lib.msolve_workspace_bytes.restype = sz
    solver_args = [vp, vp, vp, i32, dbl, i32, vp, vp, sz, vp, vp, vp, vp]
    lib.msolve_cgm.argtypes = solver_args
    lib.msolve_bicgstabm.argtypes = solver_args
    lib.msolve_multirhs_workspace_bytes.argtypes = [vp, i32, i32]
    lib.msolve_multirhs_workspace_bytes.restype = sz
    lib.msolve_solve_multirhs.argtypes = [vp, i32, vp, vp, i32, dbl, i32, vp, vp, sz, vp, vp, vp, vp]
    lib.msolve_solve_host.argtypes = [vp, i32, vp, vp, i32, dbl, i32, vp, vp, vp, vp, vp]
    lib.msolve_solve_host_batch.argtypes = [vp, i32, i32, vp, vp, i32, dbl, i32, vp, vp, vp, vp, vp]
    lib.msolve_spmv.argtypes = [vp, vp, vp, vp, vp]
    lib.msolve_profile_iteration.argtypes = [vp, i32, vp, vp, i32, i32, vp, vp, sz, vp, vp, vp]
    lib.msolve_kernel_name.argtypes = [i32, i32]
    lib.msolve_kernel_name.restype = ctypes.c_char_p
    lib.msolve_last_launch_count.argtypes = [vp]
    lib.msolve_last_launch_count.restype = i64
    lib.msolve_config.argtypes = [vp, i32, i32]
    lib.msolve_set_history.argtypes = [vp, vp, i32]
    lib.msolve_set_phase_clock.argtypes = [vp, vp]
    lib.msolve_spmv_csr_noalloc.argtypes = [ctypes.c_int64, vp, vp, vp, i32, vp, vp, vp, vp]
    lib.msolve_spmv_csr_noalloc.restype = i32
    lib.msolve_destroy.argtypes = [vp]
    lib.msolve_destroy.restype = None
    lib.msolve_last_error.restype = ctypes.c_char_p
    lib.msolve_slab_plan_create.argtypes = [ctypes.POINTER(vp), i64, i32, vp, i32, vp, vp]
    lib.msolve_slab_plan_create.restype = i32
    for name in ("msolve_slab_plan_nlocal", "msolve_slab_plan_nhalo"):
        getattr(lib, name).argtypes = [vp]
        getattr(lib, name).restype = i64
    lib.msolve_slab_plan_npeers.argtypes = [vp]
    lib.msolve_slab_plan_npeers.restype = i32
    lib.msolve_slab_plan_peer.argtypes = [vp, i32, vp, vp, vp, vp]
    lib.msolve_slab_plan_peer.restype = i32
    lib.msolve_slab_plan_colidx.argtypes = [vp]
    lib.msolve_slab_plan_colidx.restype = vp
    lib.msolve_slab_plan_destroy.argtypes = [vp]
    lib.msolve_slab_plan_destroy.restype = None
    lib.msolve_slabs_create_csr.argtypes = [ctypes.POINTER(vp), i64, i64, vp, vp, vp, i32, i32, vp, i32, vp]
    lib.msolve_slabs_create_bsr3.argtypes = [ctypes.POINTER(vp), i64, i64, vp, vp, vp, i32, i32, vp, i32, vp]
    lib.msolve_slabs_count.argtypes = [vp]
    lib.msolve_slabs_halo_elements.argtypes = [vp, i32]
    lib.msolve_slabs_halo_elements.restype = i64
    lib.msolve_slabs_workspace_bytes.argtypes = [vp, i32, i32]
    lib.msolve_slabs_workspace_bytes.restype = sz
    lib.msolve_slabs_cgm.argtypes = solver_args
    lib.msolve_slabs_bicgstabm.argtypes = solver_args
    lib.msolve_slabs_spmv.argtypes = [vp, vp, vp, vp, sz, vp, vp]
    lib.msolve_slabs_last_launch_count.argtypes = [vp]
    lib.msolve_slabs_last_launch_count.restype = i64
    lib.msolve_slabs_destroy.argtypes = [vp]
    lib.msolve_slabs_destroy.restype = None
    for name in ("msolve_slabs_create_csr", "msolve_slabs_create_bsr3", "msolve_slabs_count", "msolve_slabs_cgm",
                 "msolve_slabs_bicgstabm", "msolve_slabs_spmv"):
        getattr(lib, name).restype = i32
    for name in ("msolve_create_csr", "msolve_create_bsr3", "msolve_create_lattice_su3", "msolve_cgm", "msolve_bicgstabm",
                 "msolve_solve_host", "msolve_solve_host_batch", "msolve_spmv", "msolve_profile_iteration", "msolve_config",
                 "msolve_set_history", "msolve_set_phase_clock", "msolve_solve_multirhs"):
        getattr(lib, name).restype = i32
    _lib = lib
    return lib


def msolve_last_error() -> str:
    return load_library().msolve_last_error().decode()


def _check(rc: int) -> int:
    if rc < 0:
        raise MsolveError(rc, msolve_last_error())
    return rc


def _dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.complex64:
        return MSOLVE_C64
    if t.dtype == torch.complex128:
        return MSOLVE_C128
    if t.dtype == torch.float32:
        return MSOLVE_F32
    if t.dtype == torch.float64:
        return MSOLVE_F64
    raise TypeError("expected complex64 / complex128 / float32 / float64, got %s" % t.dtype)


def _dev(t: torch.Tensor, dtype=None) -> torch.Tensor:
    if not t.is_cuda:
        raise ValueError("expected a CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError("expected %s, got %s" % (dtype, t.dtype))
    return t.contiguous()


def _stream(stream) -> int:
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


class Matrix:
    """Owner of an `msolve_matrix*`; keeps the borrowed device arrays alive."""

    def __init__(self, handle: int, dtype: torch.dtype, n: int, keep):
        self.handle = ctypes.c_void_p(handle)
        self.dtype = dtype
        self.n = n
        self._keep = keep
        self._hist = None
        self._phase_ns = None

    def destroy(self):
        if self.handle:
            load_library().msolve_destroy(self.handle)
            self.handle = None
            self._keep = None

    def __del__(self):  # pragma: no cover
        try:
            self.destroy()
        except Exception:
            pass


def msolve_create_csr(rowptr: torch.Tensor, colidx: torch.Tensor, val: torch.Tensor,
                      flags: int = MSOLVE_SPMV_AUTO, stream=None) -> Matrix:
    lib = load_library()
    rowptr, colidx, val = _dev(rowptr, torch.int32), _dev(colidx, torch.int32), _dev(val)
    h = ctypes.c_void_p()
    n = rowptr.numel() - 1
    _check(lib.msolve_create_csr(ctypes.byref(h), n, colidx.numel(), rowptr.data_ptr(), colidx.data_ptr(),
                                 val.data_ptr(), _dtype_code(val), flags, _stream(stream)))
    return Matrix(h.value, val.dtype, n, (rowptr, colidx, val))


def msolve_create_bsr3(browptr: torch.Tensor, bcolidx: torch.Tensor, blocks: torch.Tensor,
                       flags: int = 0, stream=None) -> Matrix:
    lib = load_library()
    browptr, bcolidx, blocks = _dev(browptr, torch.int32), _dev(bcolidx, torch.int32), _dev(blocks)
    if blocks.numel() != 9 * bcolidx.numel():
        raise ValueError("blocks must hold 9 complex numbers per block")
    h = ctypes.c_void_p()
    nbrows = browptr.numel() - 1
    _check(lib.msolve_create_bsr3(ctypes.byref(h), nbrows, bcolidx.numel(), browptr.data_ptr(), bcolidx.data_ptr(),
                                  blocks.data_ptr(), _dtype_code(blocks), flags, _stream(stream)))
    return Matrix(h.value, blocks.dtype, 3 * nbrows, (browptr, bcolidx, blocks))


def msolve_create_lattice_su3(extents: Sequence[int], links: torch.Tensor, diag: float, c_f: float, c_b: float,
                              flags: int = 0, stream=None) -> Matrix:
    """Matrix-free gauged lattice operator; links[mu, s] = U_mu(s), shape (ndim, V, 3, 3)."""
    lib = load_library()
    links = _dev(links)
    ext = (ctypes.c_int32 * len(extents))(*[int(e) for e in extents])
    vol = 1
    for e in extents:
        vol *= int(e)
    if links.numel() != 9 * len(extents) * vol:
        raise ValueError("links must hold ndim * V blocks of 9 complex numbers")
    h = ctypes.c_void_p()
    _check(lib.msolve_create_lattice_su3(ctypes.byref(h), len(extents), ext, links.data_ptr(), float(diag),
                                         float(c_f), float(c_b), _dtype_code(links), flags, _stream(stream)))
    return Matrix(h.value, links.dtype, 3 * vol, (links,))


def msolve_destroy(A: Matrix) -> None:
    A.destroy()


def msolve_workspace_bytes(A: Matrix, nshifts: int, algorithm: int) -> int:
    return int(load_library().msolve_workspace_bytes(A.handle, nshifts, algorithm))


def msolve_config(A: Matrix, key: int, value: int) -> None:
    """Set option `key` (MSOLVE_CFG_*) of this handle."""
    _check(load_library().msolve_config(A.handle, key, value))


def msolve_set_history(A: Matrix, hist: Optional[torch.Tensor]) -> None:
    """Per-iteration scalar history: `hist` is a contiguous float64 CUDA tensor [cap_rows, 3 + 3 S] (CG-M) or
    [cap_rows, 8 + 6 S] (BiCGStab-M) that later solves on this handle fill row by row; None switches it off."""
    if hist is None:
        _check(load_library().msolve_set_history(A.handle, None, 0))
        A._hist = None
        return
    hist = _dev(hist, torch.float64)
    if hist.dim() != 2:
        raise ValueError("hist must be [cap_rows, row_length]")
    _check(load_library().msolve_set_history(A.handle, hist.data_ptr(), hist.shape[0]))
    A._hist = hist


def msolve_set_phase_clock(A: Matrix, ns: Optional[torch.Tensor]) -> None:
    """One-kernel path: `ns` is a contiguous int64 CUDA tensor of 16 entries that later solves on this handle add
    their per-phase nanoseconds to (include/msolve.h); None switches it off."""
    if ns is not None:
        ns = _dev(ns, torch.int64)
        if ns.numel() < 16:
            raise ValueError("ns must hold 16 entries")
    _check(load_library().msolve_set_phase_clock(A.handle, None if ns is None else ns.data_ptr()))
    A._phase_ns = ns


def msolve_last_launch_count(A: Matrix) -> int:
    return int(load_library().msolve_last_launch_count(A.handle))


@dataclass
class SolveResult:
    status: int
    iterations: int
    x: torch.Tensor            # [S, n] on the device (host tensor for msolve_solve_host)
    conv_iter: np.ndarray      # int32 [S]
    relres: np.ndarray         # float64 [S]


def _solve(fn_name: str, algorithm: int, A: Matrix, b: torch.Tensor, shifts: Sequence[float], tol: float,
           max_iter: int, x: Optional[torch.Tensor], workspace: Optional[torch.Tensor], stream) -> SolveResult:
    lib = load_library()
    b = _dev(b, A.dtype)
    if b.numel() != A.n:
        raise ValueError("b has %d elements, matrix has %d rows" % (b.numel(), A.n))
    sh = np.ascontiguousarray(shifts, dtype=np.float64)
    s = sh.size
    if x is None:
        x = torch.empty((s, A.n), dtype=A.dtype, device=b.device)
    x = _dev(x, A.dtype)
    if x.numel() != s * A.n:
        raise ValueError("x must hold nshifts*n elements")
    need = msolve_workspace_bytes(A, s, algorithm)
    if need == 0:
        raise MsolveError(MSOLVE_EINVAL, "nshifts must be in [1, %d]" % MSOLVE_MAX_SHIFTS)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=b.device)
    it = ctypes.c_int(0)
    conv = np.full(s, -1, dtype=np.int32)
    rel = np.zeros(s, dtype=np.float64)
    rc = getattr(lib, fn_name)(A.handle, b.data_ptr(), sh.ctypes.data, s, float(tol), int(max_iter), x.data_ptr(),
                               workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                               ctypes.addressof(it), conv.ctypes.data, rel.ctypes.data, _stream(stream))
    _check(rc)
    return SolveResult(rc, it.value, x.view(s, A.n), conv, rel)


def msolve_cgm(A: Matrix, b: torch.Tensor, shifts, tol: float, max_iter: int, x: Optional[torch.Tensor] = None,
               workspace: Optional[torch.Tensor] = None, stream=None) -> SolveResult:
    """CG-M (Alg. 1): solve (A + shifts[k] I) x[k] = b for every k."""
    return _solve("msolve_cgm", MSOLVE_ALG_CGM, A, b, shifts, tol, max_iter, x, workspace, stream)


def msolve_bicgstabm(A: Matrix, b: torch.Tensor, shifts, tol: float, max_iter: int, x: Optional[torch.Tensor] = None,
                     workspace: Optional[torch.Tensor] = None, stream=None) -> SolveResult:
    """BiCGStab-M."""
    return _solve("msolve_bicgstabm", MSOLVE_ALG_BICGSTABM, A, b, shifts, tol, max_iter, x, workspace, stream)


def msolve_multirhs_workspace_bytes(A: Matrix, nshifts: int, algorithm: int) -> int:
    return int(load_library().msolve_multirhs_workspace_bytes(A.handle, nshifts, algorithm))


def msolve_solve_multirhs(A: Matrix, algorithm: int, B: torch.Tensor, shifts, tol: float, max_iter: int,
                          x: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None,
                          stream=None) -> SolveResult:
    """eq. (6): (A + shifts[i] I) x[i] = B[i], one right-hand side per shift (distinct shifts)."""
    lib = load_library()
    B = _dev(B, A.dtype)
    sh = np.ascontiguousarray(shifts, dtype=np.float64)
    s = sh.size
    if B.numel() != s * A.n:
        raise ValueError("B must hold nshifts*n elements")
    if x is None:
        x = torch.empty((s, A.n), dtype=A.dtype, device=B.device)
    x = _dev(x, A.dtype)
    if x.numel() != s * A.n:
        raise ValueError("x must hold nshifts*n elements")
    need = msolve_multirhs_workspace_bytes(A, s, algorithm)
    if need == 0:
        raise MsolveError(MSOLVE_EINVAL, "nshifts must be in [1, %d]" % MSOLVE_MAX_SHIFTS)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=B.device)
    it = ctypes.c_int(0)
    conv = np.full(s, -1, dtype=np.int32)
    rel = np.zeros(s, dtype=np.float64)
    rc = lib.msolve_solve_multirhs(A.handle, algorithm, B.data_ptr(), sh.ctypes.data, s, float(tol), int(max_iter),
                                   x.data_ptr(), workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                                   ctypes.addressof(it), conv.ctypes.data, rel.ctypes.data, _stream(stream))
    _check(rc)
    return SolveResult(rc, it.value, x.view(s, A.n), conv, rel)


def msolve_solve_host(A: Matrix, algorithm: int, b: torch.Tensor, shifts, tol: float, max_iter: int,
                      x: Optional[torch.Tensor] = None, stream=None) -> SolveResult:
    """Fig. 1's call shape with HOST vectors: b and x are CPU tensors
    (pinned for full copy speed); H2D of b and D2H of all solutions happen inside the call."""
    lib = load_library()
    if b.is_cuda or b.dtype != A.dtype:
        raise ValueError("b must be a CPU tensor of the matrix dtype")
    b = b.contiguous()
    sh = np.ascontiguousarray(shifts, dtype=np.float64)
    s = sh.size
    if x is None:
        x = torch.empty((s, A.n), dtype=A.dtype, pin_memory=True)
    if x.is_cuda or x.dtype != A.dtype or x.numel() != s * A.n or not x.is_contiguous():
        raise ValueError("x must be a contiguous CPU tensor of nshifts*n elements")
    it = ctypes.c_int(0)
    conv = np.full(s, -1, dtype=np.int32)
    rel = np.zeros(s, dtype=np.float64)
    rc = lib.msolve_solve_host(A.handle, algorithm, b.data_ptr(), sh.ctypes.data, s, float(tol), int(max_iter),
                               x.data_ptr(), ctypes.addressof(it), conv.ctypes.data, rel.ctypes.data, _stream(stream))
    _check(rc)
    return SolveResult(rc, it.value, x.view(s, A.n), conv, rel)


def msolve_solve_host_batch(A: Matrix, algorithm: int, bs, shifts, tol: float, max_iter: int, xs=None, stream=None):
    """A batch of HOST right-hand sides `bs` (list of CPU tensors, pinned for overlap) -> list of SolveResult;
    the D2H copy of solution set i overlaps solve i+1 (include/msolve.h: msolve_solve_host_batch)."""
    lib = load_library()
    sh = np.ascontiguousarray(shifts, dtype=np.float64)
    s, m = sh.size, len(bs)
    bs = [b.contiguous() for b in bs]
    for b in bs:
        if b.is_cuda or b.dtype != A.dtype or b.numel() != A.n:
            raise ValueError("every b must be a CPU tensor of n elements of the matrix dtype")
    if xs is None:
        xs = [torch.empty((s, A.n), dtype=A.dtype, pin_memory=True) for _ in range(m)]
    for x in xs:
        if x.is_cuda or x.dtype != A.dtype or x.numel() != s * A.n or not x.is_contiguous():
            raise ValueError("every x must be a contiguous CPU tensor of nshifts*n elements")
    if len(xs) != m:
        raise ValueError("one x per b")
    bp = (ctypes.c_void_p * max(m, 1))(*[b.data_ptr() for b in bs])
    xp = (ctypes.c_void_p * max(m, 1))(*[x.data_ptr() for x in xs])
    it = np.zeros(max(m, 1), dtype=np.int32)
    conv = np.full((max(m, 1), s), -1, dtype=np.int32)
    rel = np.zeros((max(m, 1), s), dtype=np.float64)
    rc = lib.msolve_solve_host_batch(A.handle, algorithm, m, bp, sh.ctypes.data, s, float(tol), int(max_iter), xp,
                                     it.ctypes.data, conv.ctypes.data, rel.ctypes.data, _stream(stream))
    _check(rc)
    return [SolveResult(rc, int(it[i]), xs[i].view(s, A.n), conv[i], rel[i]) for i in range(m)]


def msolve_spmv(A: Matrix, x: torch.Tensor, y: Optional[torch.Tensor] = None, stream=None):
    """y = A x and <x, A x> (Alg. 1 l.18-19).  Returns (y, complex dot)."""
    lib = load_library()
    x = _dev(x, A.dtype)
    if y is None:
        y = torch.empty_like(x)
    dot = np.zeros(2, dtype=np.float64)
    _check(lib.msolve_spmv(A.handle, x.data_ptr(), y.data_ptr(), dot.ctypes.data, _stream(stream)))
    return y, complex(dot[0], dot[1])


MSOLVE_NOALLOC_MAX_ROWS = 1 << 20


def msolve_spmv_csr_noalloc(rowptr: torch.Tensor, colidx: torch.Tensor, val: torch.Tensor, x: torch.Tensor,
                            y: Optional[torch.Tensor] = None, dot: Optional[torch.Tensor] = None, stream=None):
    """y = A x and <x, A x> for a CSR matrix without a handle and without any device allocation inside the library
    (include/msolve.h: static scratch, n <= MSOLVE_NOALLOC_MAX_ROWS, calls that overlap on the GPU race).
    Pass `y` [n] and `dot` [2] float64 CUDA tensors to keep torch from allocating either; does not synchronise.
    Returns (y, dot) with dot = (re, im) on the device."""
    lib = load_library()
    rowptr, colidx, val = _dev(rowptr, torch.int32), _dev(colidx, torch.int32), _dev(val)
    x = _dev(x, val.dtype)
    n = rowptr.numel() - 1
    if x.numel() != n:
        raise ValueError("x must have n = rowptr.numel() - 1 entries")
    if y is None:
        y = torch.empty_like(x)
    if dot is None:
        dot = torch.empty(2, dtype=torch.float64, device=x.device)
    y, dot = _dev(y, val.dtype), _dev(dot, torch.float64)
    _check(lib.msolve_spmv_csr_noalloc(n, rowptr.data_ptr(), colidx.data_ptr(), val.data_ptr(), _dtype_code(val),
                                       x.data_ptr(), y.data_ptr(), dot.data_ptr(), _stream(stream)))
    return y, dot


def msolve_profile_iteration(A: Matrix, algorithm: int, b: torch.Tensor, shifts, iters: int,
                             x: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None, stream=None):
    """Mean per-kernel milliseconds of `iters` steady-state iterations -> {kernel name: ms}."""
    lib = load_library()
    b = _dev(b, A.dtype)
    sh = np.ascontiguousarray(shifts, dtype=np.float64)
    s = sh.size
    if x is None:
        x = torch.empty((s, A.n), dtype=A.dtype, device=b.device)
    need = msolve_workspace_bytes(A, s, algorithm)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=b.device)
    ms = np.zeros(8, dtype=np.float32)
    nl = np.zeros(8, dtype=np.int32)
    nk = _check(lib.msolve_profile_iteration(A.handle, algorithm, b.data_ptr(), sh.ctypes.data, s, int(iters),
                                             x.data_ptr(), workspace.data_ptr(), workspace.numel(),
                                             ms.ctypes.data, nl.ctypes.data, _stream(stream)))
    return {lib.msolve_kernel_name(algorithm, j).decode(): float(ms[j]) for j in range(nk)}


# ----------------------------------------------------------------------------------- row partition (slabs)
class SlabPlan:
    """Host-only plan of one slab (msolve_slab_plan_*): halo lists and renumbered columns.  No GPU involved."""

    def __init__(self, n: int, splits, rank: int, rowptr_local: np.ndarray, colidx_global: np.ndarray):
        lib = load_library()
        self._splits = np.ascontiguousarray(splits, dtype=np.int64)
        rp = np.ascontiguousarray(rowptr_local, dtype=np.int32)
        ci = np.ascontiguousarray(colidx_global, dtype=np.int32)
        h = ctypes.c_void_p()
        _check(lib.msolve_slab_plan_create(ctypes.byref(h), int(n), self._splits.size - 1, self._splits.ctypes.data,
                                           int(rank), rp.ctypes.data, ci.ctypes.data))
        self.handle = h
        self.rank = rank
        self.nlocal = int(lib.msolve_slab_plan_nlocal(h))
        self.nhalo = int(lib.msolve_slab_plan_nhalo(h))
        self.peers = []                                    # (peer rank, halo offset, global ids)
        for j in range(lib.msolve_slab_plan_npeers(h)):
            pr, off, cnt, ids = ctypes.c_int(), ctypes.c_int64(), ctypes.c_int64(), ctypes.c_void_p()
            _check(lib.msolve_slab_plan_peer(h, j, ctypes.byref(pr), ctypes.byref(off), ctypes.byref(cnt), ctypes.byref(ids)))
            arr = np.ctypeslib.as_array(ctypes.cast(ids.value, ctypes.POINTER(ctypes.c_int32)), shape=(cnt.value,)).copy() if cnt.value else np.zeros(0, np.int32)
            self.peers.append((pr.value, off.value, arr))
        nnz = int(rp[-1])
        ptr = lib.msolve_slab_plan_colidx(h)
        self.colidx = np.ctypeslib.as_array(ctypes.cast(ptr, ctypes.POINTER(ctypes.c_int32)), shape=(nnz,)).copy() if nnz else np.zeros(0, np.int32)
        lib.msolve_slab_plan_destroy(h)
        self.handle = None


class Slabs:
    """Owner of an `msolve_slabs*`: `nslabs` slabs of one matrix on the current device."""

    def __init__(self, handle, dtype, n):
        self.handle, self.dtype, self.n = ctypes.c_void_p(handle), dtype, n

    def destroy(self):
        if self.handle:
            load_library().msolve_slabs_destroy(self.handle)
            self.handle = None

    def __del__(self):  # pragma: no cover
        try:
            self.destroy()
        except Exception:
            pass


_NP2TORCH = {np.dtype(np.complex64): torch.complex64, np.dtype(np.complex128): torch.complex128,
             np.dtype(np.float32): torch.float32, np.dtype(np.float64): torch.float64}
_NP2CODE = {np.dtype(np.complex64): MSOLVE_C64, np.dtype(np.complex128): MSOLVE_C128,
            np.dtype(np.float32): MSOLVE_F32, np.dtype(np.float64): MSOLVE_F64}


def msolve_slabs_create_csr(rowptr: np.ndarray, colidx: np.ndarray, val: np.ndarray, nslabs: int, splits=None,
                            flags: int = MSOLVE_SPMV_AUTO, stream=None) -> Slabs:
    """HOST numpy arrays of the whole matrix -> `nslabs` row slabs on the current device."""
    lib = load_library()
    rp, ci, v = (np.ascontiguousarray(rowptr, dtype=np.int32), np.ascontiguousarray(colidx, dtype=np.int32),
                 np.ascontiguousarray(val))
    sp = None if splits is None else np.ascontiguousarray(splits, dtype=np.int64)
    h = ctypes.c_void_p()
    _check(lib.msolve_slabs_create_csr(ctypes.byref(h), rp.size - 1, ci.size, rp.ctypes.data, ci.ctypes.data, v.ctypes.data,
                                       _NP2CODE[v.dtype], int(nslabs), None if sp is None else sp.ctypes.data, flags, _stream(stream)))
    return Slabs(h.value, _NP2TORCH[v.dtype], rp.size - 1)


def msolve_slabs_create_bsr3(browptr: np.ndarray, bcolidx: np.ndarray, blocks: np.ndarray, nslabs: int, splits=None,
                             flags: int = MSOLVE_SPMV_AUTO, stream=None) -> Slabs:
    lib = load_library()
    rp, ci, v = (np.ascontiguousarray(browptr, dtype=np.int32), np.ascontiguousarray(bcolidx, dtype=np.int32),
                 np.ascontiguousarray(blocks))
    sp = None if splits is None else np.ascontiguousarray(splits, dtype=np.int64)
    h = ctypes.c_void_p()
    _check(lib.msolve_slabs_create_bsr3(ctypes.byref(h), rp.size - 1, ci.size, rp.ctypes.data, ci.ctypes.data, v.ctypes.data,
                                        _NP2CODE[v.dtype], int(nslabs), None if sp is None else sp.ctypes.data, flags, _stream(stream)))
    return Slabs(h.value, _NP2TORCH[v.dtype], 3 * (rp.size - 1))


def msolve_slabs_destroy(S: Slabs) -> None:
    S.destroy()


def msolve_slabs_halo_elements(S: Slabs):
    lib = load_library()
    return [int(lib.msolve_slabs_halo_elements(S.handle, p)) for p in range(lib.msolve_slabs_count(S.handle))]


def msolve_slabs_last_launch_count(S: Slabs) -> int:
    return int(load_library().msolve_slabs_last_launch_count(S.handle))


def _slabs_solve(fn_name: str, algorithm: int, S: Slabs, b, shifts, tol, max_iter, x, stream) -> SolveResult:
    lib = load_library()
    b = _dev(b, S.dtype)
    sh = np.ascontiguousarray(shifts, dtype=np.float64)
    s = sh.size
    if x is None:
        x = torch.empty((s, S.n), dtype=S.dtype, device=b.device)
    need = int(lib.msolve_slabs_workspace_bytes(S.handle, s, algorithm))
    if need == 0:
        raise MsolveError(MSOLVE_EINVAL, "nshifts must be in [1, %d]" % MSOLVE_MAX_SHIFTS)
    ws = torch.empty(need, dtype=torch.uint8, device=b.device)
    it = ctypes.c_int(0)
    conv = np.full(s, -1, dtype=np.int32)
    rel = np.zeros(s, dtype=np.float64)
    rc = getattr(lib, fn_name)(S.handle, b.data_ptr(), sh.ctypes.data, s, float(tol), int(max_iter), x.data_ptr(),
                               ws.data_ptr(), need, ctypes.addressof(it), conv.ctypes.data, rel.ctypes.data, _stream(stream))
    _check(rc)
    return SolveResult(rc, it.value, x.view(s, S.n), conv, rel)


def msolve_slabs_cgm(S: Slabs, b, shifts, tol, max_iter, x=None, stream=None) -> SolveResult:
    return _slabs_solve("msolve_slabs_cgm", MSOLVE_ALG_CGM, S, b, shifts, tol, max_iter, x, stream)


def msolve_slabs_bicgstabm(S: Slabs, b, shifts, tol, max_iter, x=None, stream=None) -> SolveResult:
    return _slabs_solve("msolve_slabs_bicgstabm", MSOLVE_ALG_BICGSTABM, S, b, shifts, tol, max_iter, x, stream)


def msolve_slabs_spmv(S: Slabs, x: torch.Tensor, stream=None):
    lib = load_library()
    x = _dev(x, S.dtype)
    y = torch.empty_like(x)
    need = int(lib.msolve_slabs_workspace_bytes(S.handle, 1, MSOLVE_ALG_CGM))
    ws = torch.empty(need, dtype=torch.uint8, device=x.device)
    dot = np.zeros(2, dtype=np.float64)
    _check(lib.msolve_slabs_spmv(S.handle, x.data_ptr(), y.data_ptr(), ws.data_ptr(), need, dot.ctypes.data, _stream(stream)))
    return y, complex(dot[0], dot[1])
