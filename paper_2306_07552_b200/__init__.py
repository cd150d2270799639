"""B200-native batch RGBD rasteriser for the rendering hot path of Galactic (arXiv 2306.07552).

`gen` (numpy only) builds the seeded synthetic workloads; `binding` is the thin ctypes layer over the
C-ABI library `libgx.so` (include/gx.h).  Importing the package loads neither torch nor the library.
"""
from importlib import import_module

__all__ = ["gen", "binding", "build"]


def __getattr__(name):
    if name in __all__:
        return import_module(f"{__name__}.{name}")
    raise AttributeError(name)
