"""delta-b200: the all-channel-pairs spectral path of the Delta framework (arxiv 2108.08896) as
hand-written CUDA for NVIDIA B200 (sm_100a) behind a C ABI (include/delta.h).

`binding` (imported lazily) loads libdelta_b200.so through ctypes; there is no CPU fallback.
"""
from . import build  # noqa: F401

__all__ = ["build", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
