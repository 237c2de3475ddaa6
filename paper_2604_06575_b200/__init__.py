"""polylab-b200: B200-native simplification of sparse multivariate polynomials.

The product is the C-ABI library built from csrc/ (include/polylab.h) and the thin
binding in `binding.py`.  Submodules load lazily so that `workloads` (pure numpy
input generators) can be imported on a box without the CUDA library; any call
into the hot path without the built library raises (there is no CPU fallback).
"""
__version__ = "0.1.0"

_LAZY = ("binding", "workloads", "build")


def __getattr__(name):
    if name in _LAZY:
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    if name in ("simplify", "mul_simplify", "simplify_host", "mul_simplify_host", "PolylabError"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
