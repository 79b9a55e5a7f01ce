"""CA-SGD outer iteration for generalized linear models, B200-native (sm_100a).

`synth` (seeded inputs) imports nothing native. Everything else goes through
`binding`, the thin ctypes layer over ``libcasgd.so`` (C ABI: include/casgd.h);
it raises at first use if the CUDA library is missing -- there is no CPU path.
"""
from . import synth  # noqa: F401

__all__ = ["synth", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
