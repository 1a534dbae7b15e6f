"""paper_2405_01834_b200: B200-native McMurchie-Davidson 3-/4-center ERI engine.

The compute path is the C-ABI library built from csrc/ (include/md_b200.h); `engine` is the thin
ctypes binding with the same names.  `workloads` holds the seeded input generators only.
There is no CPU fallback: using the engine without the built CUDA library raises.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "engine", "build"]


def __getattr__(name):
    if name in ("engine", "build"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
