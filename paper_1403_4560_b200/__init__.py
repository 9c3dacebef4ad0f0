"""B200-native Monte Carlo hot path of arXiv:1403.4560 (3D Edwards-Anderson model in a field).

`workloads` holds the seeded synthetic configs; `sg` is the thin ctypes binding over the
C-ABI library declared in include/sg.h (loaded lazily; it raises if the CUDA library has not
been built — there is no CPU fallback).
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "sg"]


def __getattr__(name):
    if name == "sg":
        import importlib
        return importlib.import_module(".sg", __name__)
    raise AttributeError(name)
