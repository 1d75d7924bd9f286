"""CPU oracle for CG-M / BiCGStab-M -- TEST INFRASTRUCTURE, NOT PRODUCT.

Thin ctypes loader around ``oracle/msolve_oracle.cpp`` (plain single-threaded C++ written
from PAPER.md; see that file's header for citations and pins).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package.  It imports nothing from ``paper_1102_2143_b200`` and shares no code with
the CUDA path.  All arrays are host numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "msolve_oracle.cpp")
_LIB = os.path.join(_HERE, "libmsolve_oracle.so")
_LIB_OMP = os.path.join(_HERE, "libmsolve_oracle_omp.so")
_lib = None
_lib_omp = None

OK, MAXITER, BREAKDOWN = 0, 1, 2
C64, C128, F32, F64 = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no fast-math, no FMA contraction, one thread)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fcx-fortran-rules", "-std=c++17",
                               "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def build_omp(force: bool = False) -> str:
    """The SAME source compiled with -fopenmp (loops over rows / elements on all host cores).  Used only by
    the timing legs of bench.py (cpu_baseline, --impl reference); never by a parity test: its dot products
    are summed per thread."""
    if force or not os.path.exists(_LIB_OMP) or os.path.getmtime(_LIB_OMP) < os.path.getmtime(_SRC):
        tmp = _LIB_OMP + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-fopenmp", "-ffp-contract=off", "-fcx-fortran-rules", "-std=c++17",
                               "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB_OMP)
    return _LIB_OMP


_ENTRY = ("oracle_spmv_csr", "oracle_cgm", "oracle_bicgstabm", "oracle_cg", "oracle_bicgstab", "oracle_multirhs")


def _load(omp: bool = False):
    global _lib, _lib_omp
    if omp:
        if _lib_omp is None:
            _lib_omp = ctypes.CDLL(build_omp())
            for name in _ENTRY:
                getattr(_lib_omp, name).restype = ctypes.c_int
        return _lib_omp
    if _lib is None:
        _lib = ctypes.CDLL(build())
        for name in _ENTRY:
            getattr(_lib, name).restype = ctypes.c_int
    return _lib


def _dt(val: np.ndarray) -> int:
    if val.dtype == np.complex64:
        return C64
    if val.dtype == np.complex128:
        return C128
    if val.dtype == np.float32:      # real: the paper's own Table 1 runs
        return F32
    if val.dtype == np.float64:
        return F64
    raise TypeError("oracle wants complex64/128 or float32/64, got %s" % val.dtype)


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _csr(rowptr, colidx, val):
    rowptr = np.ascontiguousarray(rowptr, dtype=np.int32)
    colidx = np.ascontiguousarray(colidx, dtype=np.int32)
    val = np.ascontiguousarray(val)
    return rowptr, colidx, val


def spmv(rowptr, colidx, val, x) -> np.ndarray:
    """y = A x (Alg. 1 l.18)."""
    rowptr, colidx, val = _csr(rowptr, colidx, val)
    x = np.ascontiguousarray(x, dtype=val.dtype)
    y = np.empty(rowptr.size - 1, dtype=val.dtype)
    rc = _load().oracle_spmv_csr(_dt(val), ctypes.c_int64(y.size), _p(rowptr), _p(colidx), _p(val), _p(x), _p(y))
    assert rc == 0
    return y


@dataclass
class MultishiftResult:
    status: int
    iterations: int
    x: np.ndarray           # [S, n], shift-major
    conv_iter: np.ndarray   # int32 [S]; -1 = not converged
    relres: np.ndarray      # float64 [S]: recurrence residual |zeta_k| ||r|| / ||b||
    r: np.ndarray           # base residual at exit [n]
    zeta: np.ndarray        # CG-M: float64 [S]; BiCGStab-M: complex128 [S] (= zeta_k rho_k)
    hist: Optional[np.ndarray]


def _multishift(fn_name, rowptr, colidx, val, b, shifts, tol, max_iter, stop_rule, hist_cap, hist_cols, zeta_complex,
                omp=False):
    rowptr, colidx, val = _csr(rowptr, colidx, val)
    b = np.ascontiguousarray(b, dtype=val.dtype)
    shifts = np.ascontiguousarray(shifts, dtype=np.float64)
    n, s = rowptr.size - 1, shifts.size
    x = np.empty((s, n), dtype=val.dtype)
    it = ctypes.c_int(0)
    conv = np.full(s, -1, dtype=np.int32)
    relres = np.zeros(s, dtype=np.float64)
    r = np.empty(n, dtype=val.dtype)
    zeta = np.zeros(2 * s if zeta_complex else s, dtype=np.float64)
    hist = np.zeros((hist_cap, hist_cols(s)), dtype=np.float64) if hist_cap > 0 else None
    rc = getattr(_load(omp), fn_name)(
        _dt(val), ctypes.c_int64(n), _p(rowptr), _p(colidx), _p(val), _p(b), _p(shifts), ctypes.c_int(s),
        ctypes.c_double(tol), ctypes.c_int(max_iter), ctypes.c_int(stop_rule), _p(x), ctypes.byref(it),
        _p(conv), _p(relres), _p(r), _p(zeta), _p(hist), ctypes.c_int(hist_cap))
    if rc < 0:
        raise ValueError("oracle %s: invalid arguments" % fn_name)
    if hist is not None:
        hist = hist[: min(hist_cap, it.value)]
    z = zeta.view(np.complex128) if zeta_complex else zeta
    return MultishiftResult(rc, it.value, x, conv, relres, r, z, hist)


def cgm(rowptr, colidx, val, b, shifts, tol, max_iter, stop_rule: int = 0, hist_cap: int = 0,
        omp: bool = False) -> MultishiftResult:
    """CG-M (Alg. 1, read as DESIGN.md R2-R7).  hist row = beta, alpha_next, R1,
    then zeta_new[S], beta_k[S], alpha_k[S].  stop_rule 0 = per shift (R15), 1 = literal |r| > eps (l.15).
    omp=True: the all-core build (timing legs only)."""
    return _multishift("oracle_cgm", rowptr, colidx, val, b, shifts, tol, max_iter, stop_rule,
                       hist_cap, lambda s: 3 + 3 * s, False, omp)


def bicgstabm(rowptr, colidx, val, b, shifts, tol, max_iter, stop_rule: int = 0, hist_cap: int = 0,
              omp: bool = False) -> MultishiftResult:
    """BiCGStab-M (derivation in DESIGN.md).  hist row = beta, chi, alpha' (complex), |r'|^2, 0,
    then zeta_new[S], beta_k[S], chi_k[S] (complex)."""
    return _multishift("oracle_bicgstabm", rowptr, colidx, val, b, shifts, tol, max_iter, stop_rule,
                       hist_cap, lambda s: 8 + 6 * s, True, omp)


@dataclass
class MultiRhsResult:
    status: int
    iterations: int
    x: np.ndarray           # [S, n]: x_i solves (A + sigma_i) x_i = b_i
    conv_iter: np.ndarray
    relres: np.ndarray      # |zeta_i| ||r|| / ||b_i||
    y: np.ndarray           # [S, n]: the initial guesses, b_i - (A + sigma_i) y_i = r0 for every i
    r0: np.ndarray          # [n]: the common initial residual


def multirhs(rowptr, colidx, val, B, shifts, tol, max_iter, algorithm: str = "cgm") -> MultiRhsResult:
    """A different right-hand side per shift, eq. (6): (A + shifts[i]) x[i] = B[i], through
    initial guesses with a common initial residual (S - 1 SpMVs) and ONE multishift solve."""
    rowptr, colidx, val = _csr(rowptr, colidx, val)
    shifts = np.ascontiguousarray(shifts, dtype=np.float64)
    n, s = rowptr.size - 1, shifts.size
    B = np.ascontiguousarray(B, dtype=val.dtype).reshape(s, n)
    x = np.empty((s, n), dtype=val.dtype)
    y = np.empty((s, n), dtype=val.dtype)
    r0 = np.empty(n, dtype=val.dtype)
    it = ctypes.c_int(0)
    conv = np.full(s, -1, dtype=np.int32)
    relres = np.zeros(s, dtype=np.float64)
    rc = _load().oracle_multirhs(_dt(val), ctypes.c_int64(n), _p(rowptr), _p(colidx), _p(val), _p(B), _p(shifts),
                                 ctypes.c_int(s), ctypes.c_double(tol), ctypes.c_int(max_iter),
                                 ctypes.c_int(0 if algorithm == "cgm" else 1), _p(x), ctypes.byref(it), _p(conv),
                                 _p(relres), _p(y), _p(r0))
    if rc < 0:
        raise ValueError("oracle multirhs: invalid arguments (shifts must be pairwise distinct)")
    return MultiRhsResult(rc, it.value, x, conv, relres, y, r0)


def _single(fn_name, rowptr, colidx, val, sigma, b, tol, max_iter):
    rowptr, colidx, val = _csr(rowptr, colidx, val)
    b = np.ascontiguousarray(b, dtype=val.dtype)
    n = rowptr.size - 1
    x = np.empty(n, dtype=val.dtype)
    it = ctypes.c_int(0)
    rel = ctypes.c_double(0.0)
    rc = getattr(_load(), fn_name)(_dt(val), ctypes.c_int64(n), _p(rowptr), _p(colidx), _p(val),
                                   ctypes.c_double(sigma), _p(b), ctypes.c_double(tol), ctypes.c_int(max_iter),
                                   _p(x), ctypes.byref(it), ctypes.byref(rel))
    return rc, it.value, x, rel.value


def cg(rowptr, colidx, val, sigma, b, tol, max_iter):
    """Plain CG on (A + sigma I) -- pin for CG-M.  Returns (status, iterations, x, relres)."""
    return _single("oracle_cg", rowptr, colidx, val, sigma, b, tol, max_iter)


def bicgstab(rowptr, colidx, val, sigma, b, tol, max_iter):
    """Plain BiCGStab on (A + sigma I) -- pin for BiCGStab-M."""
    return _single("oracle_bicgstab", rowptr, colidx, val, sigma, b, tol, max_iter)
