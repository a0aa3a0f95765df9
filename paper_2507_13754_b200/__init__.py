"""B200-native traditional Born series (TBS) Helmholtz solver -- hot path of arxiv 2507.13754.

The product is the CUDA library ``libtbs.so`` (C ABI in include/tbs.h); this package is its thin
binding.  Importing :mod:`paper_2507_13754_b200.tbs` requires torch; the library itself does not.
"""
from . import _lib  # noqa: F401

__all__ = ["_lib"]
