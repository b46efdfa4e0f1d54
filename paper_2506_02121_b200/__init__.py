"""B200-native critical curves and caustics of microlens fields (arXiv 2506.02121 hot path).

The product is the C-ABI library built from csrc/ (include/mlcc.h); `api` is the thin ctypes
binding with the same names.  Importing the package does not load the CUDA library; the first
call through `api` does, and fails loudly if it has not been built.
"""
from . import configs  # noqa: F401

__all__ = ["configs"]
