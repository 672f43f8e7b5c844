"""B200-native template-bank binary-pulsar search (hot path of arXiv:2112.11991).

``paper_2112_11991_b200.tb``         -- thin ctypes binding of the C-ABI in include/tb.h
                                         (loaded lazily; fails loudly if libtb.so is missing)
``paper_2112_11991_b200.workloads``  -- seeded synthetic inputs (no method arithmetic)
"""
import importlib

__all__ = ["tb", "workloads"]


def __getattr__(name):
    if name in __all__:
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
