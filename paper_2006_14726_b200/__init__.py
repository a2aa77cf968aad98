"""splat-warp for B200: the client hot path of arxiv 2006.14726 (2.5D frame -> sphere splats
-> LBVH -> ray-traced, composited reprojection) as hand-written sm_100a CUDA kernels behind
the C ABI of include/splats.h.  `binding` holds the ctypes wrappers (same names as the C
calls); `build` compiles the shared library in-tree."""
from . import build  # noqa: F401

__all__ = ["build", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
