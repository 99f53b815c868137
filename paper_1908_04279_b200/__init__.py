"""paper_1908_04279_b200 -- B200-native bound-motor microscale step (after arxiv 1908.04279).

The product is libmm.so (hand-written CUDA for sm_100a behind the C ABI of include/mm.h); this package
is its build script and a thin ctypes binding.  No CPU fallback exists.
"""
from .binding import MM, MMError, lib  # noqa: F401
from . import binding, build  # noqa: F401
