"""B200-native Splotch render hot path (arxiv 1004.1302): C-ABI CUDA library + thin binding.

    from paper_1004_1302_b200 import binding   # ctypes face of include/splotch.h
    from paper_1004_1302_b200 import Scene     # device residency + one-call renders

Importing the package does not load the CUDA library; the first call does, and fails loudly if
libsplotch_b200.so has not been built (python -m paper_1004_1302_b200.build).  No CPU fallback.
"""
from . import binding  # noqa: F401


def __getattr__(name):
    if name == "Scene":
        from .scene import Scene
        return Scene
    raise AttributeError(name)
