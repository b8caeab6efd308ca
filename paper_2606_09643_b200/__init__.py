"""paper_2606_09643_b200 — B200-native mixed-task vFM forward (FMplex deployment sharing).

The product is libfmx.so (CUDA kernels for sm_100a behind the C ABI in include/fmx.h).
This package holds its sources (csrc/), the build step, a thin ctypes binding with the same
names, and a Session helper that uploads a seeded workload.  There is no CPU fallback: without
the built library `binding.load()` raises, and without a B200 `fmx_create` fails.
"""
from .binding import Fmx, Bfq, FmxError, load, LIB_PATH  # noqa: F401

__all__ = ["Fmx", "Bfq", "FmxError", "load", "LIB_PATH"]
