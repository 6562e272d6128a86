"""B200-native SLDG hot path of arxiv 2212.03036: thin Python binding over the C-ABI library libsldg.

The compute lives entirely in paper_2212_03036_b200/csrc (CUDA, sm_100a) behind include/sldg.h; this
package only marshals arguments.  PyTorch is used by callers for device memory and streams.
Importing the package is cheap; the shared library is loaded on first use and the product path fails
loudly when it is missing or no CUDA device is present.
"""
import importlib

from . import inputs  # noqa: F401  (seeded generators, no arithmetic of the method)

__all__ = ["inputs", "binding", "Sldg", "SldgError"]


def __getattr__(name):
    if name == "binding":
        return importlib.import_module(__name__ + ".binding")
    if name in ("Sldg", "SldgError", "load_library"):
        return getattr(importlib.import_module(__name__ + ".binding"), name)
    raise AttributeError(name)
