"""Regression of the oracle against the stored golden values (written by
tests/golden/make_golden.py from the oracle alone), and the GPU against the same values."""
import json
import os

import numpy as np
import pytest

import oracle
from paper_1102_2143_b200 import workloads as W

GOLDEN = json.load(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "iteration_counts.json")))

CASES = {
    "config1": lambda: W.config1(),
    "config2": lambda: W.config2(),
    "config3_8x8x8x8": lambda: W.config3(extents=(8, 8, 8, 8)),
    "config4_8x8x8x16": lambda: W.config4(extents=(8, 8, 8, 16)),
    "config4_8x8x8x16_c64": lambda: W.config4(extents=(8, 8, 8, 16), tol=1e-5),
    "config5_n16384": lambda: W.config5(n=1 << 14),
}


def _dtype(name):
    return np.complex64 if name.endswith("c64") else np.complex128


@pytest.mark.parametrize("name", ["config1", "config3_8x8x8x8", "config4_8x8x8x16_c64"])
def test_oracle_reproduces_golden(name):
    w = CASES[name]()
    fn = oracle.cgm if w.algorithm == "cgm" else oracle.bicgstabm
    dt = _dtype(name)
    r = fn(w.rowptr, w.colidx, w.val.astype(dt), w.b.astype(dt), w.shifts, w.tol, w.max_iter)
    g = GOLDEN[name]
    assert r.status == g["status"] and r.iterations == g["iterations"]
    assert list(r.conv_iter) == g["conv_iter"]
    assert abs(np.linalg.norm(r.x[0].astype(np.complex128)) - g["x0_norm"]) <= 1e-6 * g["x0_norm"]


@pytest.mark.gpu
@pytest.mark.parametrize("name", sorted(CASES))
def test_gpu_iteration_counts_vs_golden(name):
    import torch
    from paper_1102_2143_b200 import binding as ms, build
    build.build()
    w = CASES[name]()
    dt = _dtype(name)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()  # noqa: E731
    if w.has_bsr3:
        A = ms.msolve_create_bsr3(dev(w.browptr), dev(w.bcolidx), dev(w.blocks.astype(dt)))
    else:
        A = ms.msolve_create_csr(dev(w.rowptr), dev(w.colidx), dev(w.val.astype(dt)))
    fn = ms.msolve_cgm if w.algorithm == "cgm" else ms.msolve_bicgstabm
    r = fn(A, dev(w.b.astype(dt)), w.shifts, w.tol, w.max_iter)
    g = GOLDEN[name]
    assert r.status == g["status"]
    assert abs(r.iterations - g["iterations"]) <= 2
    assert np.all(np.abs(r.conv_iter - np.array(g["conv_iter"])) <= 2)
    x0 = torch.linalg.vector_norm(r.x[0].to(torch.complex128)).item()
    assert abs(x0 - g["x0_norm"]) <= 1e-4 * g["x0_norm"]
    ms.msolve_destroy(A)
