"""B200-native GOTHIC hot path (arxiv 1610.07279): oct-tree build, block time-step bookkeeping and the
gravity walk for the active i-particles, as hand-written sm_100a CUDA behind the C ABI of include/gothic.h.

`workloads` (seeded synthetic inputs) is importable anywhere; `binding` needs the in-tree
libgothic_b200.so and a CUDA device and raises GothicError otherwise (there is no CPU fallback)."""
import importlib

from . import workloads  # noqa: F401

__all__ = ["workloads", "Gothic", "GothicError", "load_library"]


def __getattr__(name):
    if name in ("Gothic", "GothicError", "load_library"):
        return getattr(importlib.import_module(".binding", __name__), name)
    raise AttributeError(name)
