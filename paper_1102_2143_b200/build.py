"""Build libmsolve.so (the C-ABI library of include/msolve.h) in-tree with nvcc for sm_100a.

The library is several translation units (csrc/handle.h lists them); they are compiled in parallel into
csrc/../build/*.o and linked into one shared object.  spmv_role.cu is compiled once per SpMV role."""
from __future__ import annotations

import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libmsolve.so")
# (source, object name, extra defines)
UNITS = [("msolve.cu", "msolve.o", []), ("vec.cu", "vec.o", []), ("fused_small.cu", "fused_small.o", []),
         ("slab.cu", "slab.o", []), ("multirhs.cu", "multirhs.o", []), ("resident.cu", "resident.o", []),
         ("noalloc.cu", "noalloc.o", [])] + \
        [("spmv_role.cu", "spmv_role%d.o" % r, ["-DMSOLVE_ROLE=%d" % r]) for r in range(4)]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-Xptxas", "-v",
]


def _inputs():
    files = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh", ".h"))]
    return files + [os.path.join(HERE, "..", "include", "msolve.h"), os.path.abspath(__file__)]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in _inputs())


def _compile(nvcc, src, obj, defs):
    cmd = [nvcc] + NVCC_FLAGS + defs + ["-c", "-o", obj, os.path.join(CSRC, src)]
    proc = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    return src, defs, proc.returncode, proc.stdout


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or stale()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    tag = ".tmp%d" % os.getpid()
    units = [(s, os.path.join(OBJ, "p%d_" % os.getpid() + o), d) for s, o, d in UNITS if os.path.exists(os.path.join(CSRC, s))]
    log = []
    failed = False
    with concurrent.futures.ThreadPoolExecutor(max_workers=min(len(units), os.cpu_count() or 1)) as pool:
        for src, defs, rc, out in pool.map(lambda u: _compile(nvcc, *u), units):
            log.append("==== %s %s\n%s" % (src, " ".join(defs), out))
            if rc != 0:
                failed = True
                sys.stderr.write(out)
    if verbose and not failed:
        sys.stderr.write("\n".join(log))
    try:
        if failed:
            raise RuntimeError("nvcc failed")
        tmp = LIB + tag
        cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static", "-o", tmp] + [u[1] for u in units]
        proc = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        if proc.returncode != 0:
            sys.stderr.write(proc.stdout)
            raise RuntimeError("link failed (exit %d)" % proc.returncode)
        with open(os.path.join(HERE, "build_ptxas.log"), "w") as f:
            f.write("\n".join(log))
        os.replace(tmp, LIB)
    finally:
        for _, o, _ in units:
            if os.path.exists(o):
                os.remove(o)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
