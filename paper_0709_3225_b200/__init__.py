"""B200-native Lennard-Jones MD hot path of arXiv 0709.3225 (velocity Verlet with
all-pairs and cell-list forces, rand48 with skip-ahead).

The product is the C-ABI library declared in include/ljmd.h and built from csrc/;
`binding` is a thin ctypes layer with the same names.  Importing `binding` (or any
name re-exported from it) raises if the CUDA library has not been built: there is
no CPU fallback.  `workloads` (input generators only) imports without it.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding", "build"]


def __getattr__(name):
    if name in ("binding", "build"):
        import importlib
        return importlib.import_module("." + name, __name__)
    raise AttributeError(name)
