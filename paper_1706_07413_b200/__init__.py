"""adsc — batched AdS4 scalar-collapse RK4 stepper for B200 (sm_100a).

Thin Python binding over the C-ABI library libadsc.so (include/adsc.h).  The
binding only marshals arguments; every step of the path runs in the CUDA
kernels under csrc/.  Importing this package does not load the library;
the first use does, and fails loudly if it is missing (no CPU fallback).
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "Ensemble", "load_library", "AdscError"]


def __getattr__(name):
    if name in ("Ensemble", "load_library", "AdscError", "adsc_diag"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
