"""B200-native hot path of Kamera's training-free KV-reuse operator (arxiv/paper_2606_23581).

The product is libkamera.so (C ABI in include/kamera.h, CUDA for sm_100a in csrc/); this package is its thin
ctypes binding.  Nothing here computes: if the library cannot be built/loaded, calls raise.
"""
from .binding import *          # noqa: F401,F403
from .binding import lib, Context, Pool, Chunk, Patch, make_layout, patch_refs, KameraError   # noqa: F401
