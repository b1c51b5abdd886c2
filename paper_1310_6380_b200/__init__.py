"""B200-native hot path of the mixed-variational phononic band-structure method (arXiv:1310.6380).

``libbs.so`` (hand-written sm_100a CUDA behind the C-ABI of ``include/bs.h``) does all the work; this package is the
thin ctypes binding with the same names.  No CPU fallback exists: the binding is loaded on first attribute access and
raises ``ImportError`` when ``libbs.so`` has not been built (``python -m paper_1310_6380_b200.build``).
"""
import importlib

__all__ = ["binding", "build"]


def __getattr__(name):
    # lazy so that ``python -m paper_1310_6380_b200.build`` can run before the library exists
    if name.startswith("__"):
        raise AttributeError(name)
    binding = importlib.import_module(".binding", __name__)
    try:
        return getattr(binding, name)
    except AttributeError:
        raise AttributeError(f"module {__name__!r} has no attribute {name!r}") from None
