"""dmx — B200-native batched adaptive-step contact rollouts with CFD gradients (arxiv 2506.14186).

`workloads` (seeded input generation) imports without a GPU; everything else goes through the
CUDA C-ABI library and fails loudly when it is missing.
"""
import importlib

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name in __all__:
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
