"""B200-native fp64 electromagnetic particle-in-cell hot path (gather, Boris
push, Esirkepov deposition, Yee FDTD, per-cell counting sort) behind a C-ABI
library.  ``Sim`` is the thin binding; ``workloads`` holds the seeded inputs.

The compute path is the CUDA library only: there is no CPU fallback, and
``Sim`` raises if ``libpic_b200.so`` is missing."""
from . import workloads  # noqa: F401

__all__ = ["workloads", "Sim", "PicError", "load_library", "build_library"]


def __getattr__(name):
    if name in ("Sim", "PicError", "load_library", "LIB_PATH"):
        from . import binding
        return getattr(binding, name)
    if name == "build_library":
        from .build import build_library
        return build_library
    raise AttributeError(name)
