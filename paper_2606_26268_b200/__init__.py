"""paper_2606_26268_b200 — B200-native gray-M1 radiation sub-step (arxiv 2606.26268, Sect. 2.4-2.8).

The product is the C-ABI CUDA library `librt_m1.so` (include/rt.h, csrc/); `rt` is its thin ctypes
binding.  Importing the package does not need a GPU; calling into it does (no CPU path).
"""
from . import build  # noqa: F401

__all__ = ["build", "rt"]


def __getattr__(name):
    if name == "rt":
        import importlib
        return importlib.import_module(".rt", __name__)
    raise AttributeError(name)
