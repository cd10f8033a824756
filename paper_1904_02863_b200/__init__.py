"""B200-native batched TaylorF2 waveform + Gaussian likelihood (arXiv:1904.02863 hot path).

``inputs`` is importable anywhere (numpy only).  The CUDA binding (``GwContext`` and the
``gw_*`` entry points of include/gwlnl.h) is imported lazily and fails loudly when the
extension ``csrc/libgwlnl.so`` is missing: there is no CPU fallback.
"""
from . import inputs  # noqa: F401

_LAZY = ("binding", "GwContext", "GwError", "lib_path", "load_library")


def __getattr__(name):
    if name in _LAZY:
        import importlib
        mod = importlib.import_module(".binding", __name__)
        return mod if name == "binding" else getattr(mod, name)
    raise AttributeError(name)
