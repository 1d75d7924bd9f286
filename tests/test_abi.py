"""The C-ABI library loads and exports every symbol include/msolve.h declares (no GPU needed),
and argument validation that happens before any CUDA call."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1102_2143_b200 import build, binding
    build.build()
    return binding.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "msolve.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(msolve_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_all_exported(lib):
    names = _declared_symbols()
    assert "msolve_cgm" in names and "msolve_bicgstabm" in names and "msolve_create_bsr3" in names
    for name in names:
        assert hasattr(lib, name), "libmsolve.so does not export %s" % name


def test_binding_export_list_matches_header():
    from paper_1102_2143_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_symbols()


def test_validation_without_gpu(lib):
    # these return before touching CUDA
    h = ctypes.c_void_p()
    assert lib.msolve_create_csr(ctypes.byref(h), -1, 0, None, None, None, 1, 0, None) == -1
    assert b"bad n/nnz" in lib.msolve_last_error()
    assert lib.msolve_create_csr(ctypes.byref(h), 4, 4, None, None, None, 1, 0, None) == -1
    assert lib.msolve_create_bsr3(ctypes.byref(h), 4, 4, None, None, None, 7, 0, None) == -1
    ext = (ctypes.c_int32 * 4)(4, 4, 4, 4)
    assert lib.msolve_create_lattice_su3(ctypes.byref(h), 5, ext, None, 8.0, 1.0, 1.0, 1, 0, None) == -1
    assert b"ndim" in lib.msolve_last_error()
    assert lib.msolve_create_lattice_su3(ctypes.byref(h), 4, ext, None, 8.0, 1.0, 1.0, 1, 0, None) == -1
    assert lib.msolve_workspace_bytes(None, 4, 0) == 0
    assert lib.msolve_config(None, 0, 0) == -1
    assert lib.msolve_set_history(None, None, 0) == -1
    assert lib.msolve_set_phase_clock(None, None) == -1
    # the solver entry points and the profiler check the handle before anything else
    sh = (ctypes.c_double * 1)(0.0)
    for fn in (lib.msolve_cgm, lib.msolve_bicgstabm):
        assert fn(None, None, sh, 1, 1e-10, 10, None, None, 0, None, None, None, None) == -1
        assert b"A is NULL" in lib.msolve_last_error()
    ms_buf = (ctypes.c_float * 8)()
    assert lib.msolve_profile_iteration(None, 0, None, sh, 1, 1, None, None, 0, ms_buf, None, None) == -1
    assert lib.msolve_solve_host(None, 0, None, sh, 1, 1e-10, 10, None, None, None, None, None) == -1
    assert lib.msolve_spmv(None, None, None, None, None) == -1
    assert lib.msolve_last_launch_count(None) == 0
    assert lib.msolve_kernel_name(0, 1) == b"spmv_dot"
    lib.msolve_destroy(None)  # no-op


def test_no_oracle_reference_in_product():
    # the product path must not import, link or execute anything under oracle/
    pkg = os.path.join(ROOT, "paper_1102_2143_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "msolve_oracle" not in src, f
