"""B200-native fp64 curvilinear Navier–Stokes RHS + RK-stage hot path (arxiv 2006.07964).

`workloads` (seeded synthetic inputs) is importable without the CUDA library; every other name
is resolved lazily from `.binding`, which loads the C-ABI shared library and raises loudly when it
is missing (there is no CPU fallback).
"""
from . import workloads  # noqa: F401

_BINDING_NAMES = ("Context", "CfdError", "lib", "LIB_PATH", "NG", "device_peak_probe")


def __getattr__(name):
    if name == "binding" or name in _BINDING_NAMES:
        import importlib

        b = importlib.import_module(".binding", __name__)
        return b if name == "binding" else getattr(b, name)
    raise AttributeError(name)
