"""B200-native RFA bioheat stepping (arXiv 1907.05709 hot path).

``workloads`` (seeded synthetic inputs) is importable everywhere.  The simulation class ``RfaSim`` is a
thin ctypes binding over the C-ABI CUDA library ``librfa.so``; it is imported lazily so that CPU-only
tooling can use the input generators, and it raises if the library has not been built.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "RfaSim", "load_library"]


def __getattr__(name):
    if name in ("RfaSim", "load_library", "RfaError", "binding"):
        from . import binding
        return binding if name == "binding" else getattr(binding, name)
    raise AttributeError(name)
