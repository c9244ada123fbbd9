"""B200-native hot path of accLB (arXiv 2505.01126): the per-time-step lattice update.

``binding``   thin ctypes layer over the C-ABI library ``libacclb.so`` (include/acclb.h); every step of the path
              runs in the hand-written sm_100a kernels under ``csrc/``.  There is no CPU fallback.
``workloads`` seeded synthetic inputs (numpy only, none of the method's arithmetic).
"""
from importlib import import_module

__all__ = ["binding", "workloads", "build"]


def __getattr__(name):
    if name in __all__:
        return import_module(f"{__name__}.{name}")
    raise AttributeError(name)
