"""B200-native hot path of arXiv:2304.09139: dd-accurate stealthy energy, gradient, S_max, minimizer.

``paper_2304_09139_b200.shd`` is the thin ctypes binding over the C-ABI library (include/shd.h);
it is imported lazily so that ``inputs`` (pure numpy workload recipes) stays importable on a
machine without the built library.  There is no CPU fallback: using ``shd`` without
``libshd.so`` raises.
"""
__all__ = ["inputs", "shd"]


def __getattr__(name):
    if name in ("shd", "inputs"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
