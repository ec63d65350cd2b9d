"""B200-native TDVP hot path of arXiv:1907.12044 (H_eff apply, environment updates, TDVP-PS / TDVP-MU
step drivers) as a C-ABI CUDA library (include/tdvp.h, csrc/) plus a thin ctypes binding.

`paper_1907_12044_b200.build` compiles libtdvp.so; every other name is served from `.binding`,
which loads the library on first use and raises when it is missing (there is no CPU fallback).
"""
import importlib

_BINDING = None


def __getattr__(name):
    global _BINDING
    if name.startswith("__"):
        raise AttributeError(name)
    if name in ("build", "binding"):
        return importlib.import_module("." + name, __name__)
    if _BINDING is None:
        _BINDING = importlib.import_module(".binding", __name__)
    return getattr(_BINDING, name)
