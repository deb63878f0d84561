"""B200-native (sm_100a) implementation of the PyDoseRT dose hot path (arxiv 2512.18863).

`Engine` wraps the C ABI of include/pdrt.h (libpdrt.so: hand-written CUDA kernels); `workloads` holds the
seeded synthetic inputs.  Importing the package does not touch CUDA; creating an Engine does, and fails
loudly when the library is not built or no GPU is present (there is no CPU fallback).
"""
from . import workloads  # noqa: F401
from .binding import Engine, PdrtError, PdrtLimits, load_library, LIB_PATH, SYMBOLS, STAGES  # noqa: F401
