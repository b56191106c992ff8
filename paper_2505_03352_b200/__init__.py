"""epsgrad: B200-native C -> eps_hat (Yee grid) chain and its Eq. (1) reverse pass.

The product is the C-ABI library built from ``csrc/`` (``include/epsgrad.h``);
``binding`` is the thin ctypes layer over it.  Nothing here imports the oracle.
The CUDA library is loaded on first use and its absence is a hard error.
"""
from . import workloads  # noqa: F401  (pure-numpy input recipes; no CUDA needed)

__all__ = ["workloads", "binding", "build"]


def __getattr__(name):
    if name in ("binding", "build"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
