"""B200-native multishift Krylov solvers CG-M / BiCGStab-M (arXiv 1102.2143).

`binding` mirrors the C ABI of include/msolve.h over libmsolve.so (hand-written sm_100a
kernels); `workloads` holds the seeded input generators; `build` compiles the library in-tree.
Nothing here computes on the CPU: without the CUDA library every solver call raises.
"""
from . import workloads  # noqa: F401  (pure numpy, safe without a GPU)

__all__ = ["workloads", "binding", "build"]


def __getattr__(name):
    if name in ("binding", "build"):
        import importlib
        return importlib.import_module("." + name, __name__)
    raise AttributeError(name)
