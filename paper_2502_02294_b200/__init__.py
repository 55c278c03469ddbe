"""diffHydro coupled hydro + particle-mesh step and its adjoint, hand-written CUDA for sm_100a (B200).

`workloads` (numpy input recipes) imports without the CUDA library; `api` (the thin ctypes binding over the
C-ABI library libdiffhydro.so) raises ImportError loudly when the library has not been built -- there is no CPU
fallback anywhere in this package.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "api"]


def __getattr__(name):
    if name == "api":
        import importlib
        return importlib.import_module(".api", __name__)
    raise AttributeError(name)
