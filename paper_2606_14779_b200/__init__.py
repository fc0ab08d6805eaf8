"""kvpool — B200-native unified KV pooling hot path (arxiv 2606.14779).

`workloads` (seeded synthetic inputs) imports nothing native.  Everything else lives in `binding`
(ctypes over the C ABI declared in include/kvpool.h) and is loaded lazily on first attribute access;
there is no CPU fallback — a missing libkvpool.so raises.
"""
from importlib import import_module

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name in ("workloads", "binding", "build"):
        return import_module(f"{__name__}.{name}")
    binding = import_module(f"{__name__}.binding")
    try:
        return getattr(binding, name)
    except AttributeError:
        raise AttributeError(f"module {__name__!r} has no attribute {name!r}") from None
