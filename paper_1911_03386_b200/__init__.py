"""B200-native ensemble Cahn-Hilliard ADI stepper (arXiv 1911.03386 hot path).

`inputs` is the seeded synthetic-input module (shared with the oracle, no arithmetic
of the method); `binding` is the thin ctypes layer over the C ABI in include/ch.h.
Nothing here falls back to a CPU implementation: using the binding without the
compiled CUDA library raises.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
