"""B200-native fused attention + JVP under frame/chunk masks (arxiv/paper_2606_25473, App. B).

The product is the C-ABI library `libattn_jvp.so` (include/attn_jvp.h); `binding` exposes the same entry
points to Python.  Importing `binding` members loads the library and raises if it has not been built:
there is no CPU or PyTorch fallback path.
"""
from . import workloads  # noqa: F401  (shapes and seeded random inputs only)

__all__ = ["binding", "workloads", "build"]


def __getattr__(name):
    if name in ("binding", "build"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
