"""B200-native hot path of LOC line radiative transfer (arxiv 2009.12609): C-ABI CUDA library + thin binding.

    from paper_2009_12609_b200 import binding, LocModel

`binding` mirrors include/loc.h one to one; `LocModel` owns the device buffers of a model.  There is no CPU
implementation in this package (the float64 oracle under oracle/ is test infrastructure and is never imported here).
"""


def __getattr__(name):  # lazy: model.py imports torch, binding.py loads the shared library
    if name == "LocModel":
        from .model import LocModel
        return LocModel
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
