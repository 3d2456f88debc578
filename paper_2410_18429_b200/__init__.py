"""paper_2410_18429_b200 — B200-native batched LSQR for 3D wavefield reconstruction inversion.

The product is libwri.so (CUDA, sm_100a; C ABI in include/wri.h).  This package is the thin
Python binding: argument marshalling only.  PyTorch supplies device memory and streams.
There is no CPU fallback: without the built library or without a CUDA device every compute
entry raises.
"""
from .binding import Wri, WriError, lib_path, load_library  # noqa: F401
