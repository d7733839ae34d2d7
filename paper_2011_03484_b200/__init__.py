"""B200-native GLISSE hot path (arXiv 2011.03484): test-particle Wisdom–Holman integrator.

The product is the C-ABI library built from csrc/ (include/glisse.h); `binding` is the thin
ctypes layer over it and `inputs` the seeded workload generators.  Submodules are loaded lazily so
that `paper_2011_03484_b200.inputs` can be imported without the CUDA library being present.
"""
import importlib

__all__ = ["binding", "inputs", "build"]


def __getattr__(name):
    if name in __all__:
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
