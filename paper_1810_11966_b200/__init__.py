"""B200-native first-level J/psi trigger for the CBM muon chambers (arxiv 1810.11966).

The product is the C-ABI library ``libcbmtrigger.so`` (include/cbm_trigger.h) built from
``csrc/``; ``binding`` is its thin ctypes binding.  Nothing here falls back to the CPU: if
the CUDA library is missing, the binding raises.
"""
from . import workloads  # noqa: F401  (input generators only)

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
