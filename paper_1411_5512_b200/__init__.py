"""B200-native checkerboard Metropolis engine for the 3D +-J Edwards-Anderson model.

The product is the C-ABI library built from `csrc/` (declared in include/ea.h); `binding`
is a thin ctypes marshalling layer with the same names.  Importing the package is cheap;
the shared library is loaded on first use and a missing library raises (there is no CPU
fallback of any kind).
"""
from . import workloads  # noqa: F401  (no method arithmetic in there)

__all__ = ["workloads", "binding", "build"]


def __getattr__(name):
    if name in ("binding", "build"):
        import importlib
        return importlib.import_module("." + name, __name__)
    raise AttributeError(name)
