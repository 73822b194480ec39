"""B200-native DPSR layer (Shape As Points, arXiv 2106.03452): hand-written sm_100a kernels
behind the C ABI in include/sap_dpsr.h.  Importing the package is cheap; the CUDA library is
loaded on first use and its absence is an error (there is no CPU fallback)."""
import importlib

__all__ = ["inputs", "binding", "Dpsr", "dpsr"]


def __getattr__(name):
    if name in ("Dpsr", "dpsr"):
        return getattr(importlib.import_module(".binding", __name__), name)
    raise AttributeError(name)
