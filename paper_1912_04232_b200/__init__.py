"""B200-native neighbor-list molecular-dynamics hot path (arXiv 1912.04232).

The product is the C-ABI library ``libmd_b200.so`` (``include/md.h``,
``csrc/``); ``binding`` is the thin ctypes layer over it with the same names.
Nothing here falls back to a CPU implementation: calling any compute entry
point without the built CUDA library raises.
"""
from . import workloads  # noqa: F401  (pure NumPy; no CUDA needed)

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
