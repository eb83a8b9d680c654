"""hpmc-b200: B200-native checkerboard Metropolis sweep for hard shapes (arXiv:1509.04692).

`workloads` (numpy only) builds the seeded synthetic inputs; everything else is the thin ctypes
binding over the hand-written CUDA library `libhpmc.so` (C-ABI in include/hpmc.h) and is loaded
lazily so that `import paper_1509_04692_b200.workloads` needs neither torch nor the library.
There is no CPU fallback: using the binding without the built library raises.
"""
import importlib

__all__ = ["workloads", "binding", "Hpmc", "build"]


def __getattr__(name):
    if name in ("workloads", "binding", "build"):
        return importlib.import_module(f"{__name__}.{name}")
    if name == "Hpmc":
        return importlib.import_module(f"{__name__}.binding").Hpmc
    raise AttributeError(name)
