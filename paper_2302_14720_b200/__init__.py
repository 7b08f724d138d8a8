"""Swendsen-Wang sweep for the 2D periodic Ising model on one NVIDIA B200 (sm_100a).

The product is the CUDA library under ``csrc/`` behind the C ABI of ``include/sw.h``;
``binding`` is the thin ctypes layer with the same names.  There is no CPU fallback:
using the binding without the built ``libsw_b200.so`` raises.
"""
from importlib import import_module as _imp

__all__ = ["binding", "workloads", "build"]


def __getattr__(name):
    if name in __all__:
        return _imp(f"{__name__}.{name}")
    raise AttributeError(name)
