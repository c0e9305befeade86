"""rmsynth-b200: Faraday rotation-measure synthesis (arxiv 1810.06250) on one NVIDIA B200.

The product is the C-ABI library librmsynth.so (include/rmsynth.h); `binding` is a thin
ctypes layer with the same entry-point names.  Import of the binding is lazy so that
`paper_1810_06250_b200.build` can be used before the library exists.
"""
__all__ = ["binding", "build"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
