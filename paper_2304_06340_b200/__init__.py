"""B200-native hot path of arXiv 2304.06340 (weak distance between S^2 and its triangulations): the Fourier
transform of a triangle-mesh surface measure on a ball-shaped frequency quadrature and the H^{-s} distance to the
unit sphere.  Hand-written CUDA for sm_100a behind the C ABI of include/sfd.h; this package is its ctypes binding.

The binding is loaded on first attribute access (so that `paper_2304_06340_b200.build` can be imported to compile
libsfd.so before it exists); if the library is missing that access raises ImportError -- there is no fallback.
"""
import importlib

_binding = None


def _load():
    global _binding
    if _binding is None:
        _binding = importlib.import_module(".binding", __name__)
    return _binding


def __getattr__(name):
    if name.startswith("__"):
        raise AttributeError(name)
    if name in ("build", "binding"):
        return importlib.import_module("." + name, __name__)
    b = _load()
    try:
        return getattr(b, name)
    except AttributeError:
        raise AttributeError(f"module {__name__!r} has no attribute {name!r}") from None


def __dir__():
    return sorted(set(globals()) | set(dir(_load())))
