"""B200-native RFA bioheat stepping (arXiv 1907.05709 hot path).

``workloads`` (seeded synthetic inputs) is importable everywhere.  The simulation class ``RfaSim`` is a
thin ctypes binding over the C-ABI CUDA library ``librfa.so``; it is resolved lazily so that CPU-only
tooling can use the input generators, and it raises if the library has not been built.
"""
import importlib

from . import workloads  # noqa: F401

__all__ = ["workloads", "RfaSim", "RfaError", "load_library", "from_workload"]


def __getattr__(name):
    if name in ("RfaSim", "RfaError", "load_library", "from_workload"):
        return getattr(importlib.import_module(".binding", __name__), name)
    raise AttributeError(name)
