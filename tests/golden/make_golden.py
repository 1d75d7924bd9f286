"""Writes tests/golden/iteration_counts.json from the CPU oracle ONLY (never from the CUDA path).

    python tests/golden/make_golden.py

The paper prints no worked numerical example, so these are regression
values of the pinned oracle on the seeded BASELINE configs (scaled where the full size takes long),
used to (a) detect drift of the oracle or the generators and (b) bound the GPU's iteration counts.
"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import oracle  # noqa: E402
from paper_1102_2143_b200 import workloads as W  # noqa: E402

CASES = {
    "config1": lambda: W.config1(),
    "config2": lambda: W.config2(),
    "config3_8x8x8x8": lambda: W.config3(extents=(8, 8, 8, 8)),
    "config4_8x8x8x16": lambda: W.config4(extents=(8, 8, 8, 16)),
    "config4_8x8x8x16_c64": lambda: W.config4(extents=(8, 8, 8, 16), tol=1e-5),
    "config5_n16384": lambda: W.config5(n=1 << 14),
}


def main():
    out = {}
    for name, make in CASES.items():
        w = make()
        dtype = np.complex64 if name.endswith("c64") else np.complex128
        fn = oracle.cgm if w.algorithm == "cgm" else oracle.bicgstabm
        r = fn(w.rowptr, w.colidx, w.val.astype(dtype), w.b.astype(dtype), w.shifts, w.tol, w.max_iter)
        out[name] = {"algorithm": w.algorithm, "n": int(w.n), "tol": w.tol, "status": int(r.status),
                     "iterations": int(r.iterations), "conv_iter": [int(c) for c in r.conv_iter],
                     "x0_norm": float(np.linalg.norm(r.x[0].astype(np.complex128)))}
        print(name, out[name]["iterations"], out[name]["conv_iter"])
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "iteration_counts.json"), "w") as f:
        json.dump(out, f, indent=1)


if __name__ == "__main__":
    main()
