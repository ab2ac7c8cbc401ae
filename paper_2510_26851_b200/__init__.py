"""B200-native periodic Friends-of-Friends (the hot path of jFoF, arxiv 2510.26851).

`binding` holds the thin ctypes/torch marshalling over the C ABI of include/fof.h
(libfof_b200.so, hand-written sm_100a CUDA).  `inputs` holds the seeded synthetic workloads.
Nothing is loaded at import time; the first binding call loads the shared library and raises
if it is missing — there is no CPU fallback.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib

        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
