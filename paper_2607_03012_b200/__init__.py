"""B200-native HyperVAttention operator (arxiv/paper_2607_03012): CUDA kernels behind the C ABI of
include/hva.h (`libhva.so`), a ctypes binding with the same names (`binding`), and the seeded
workload generator (`inputs`).  The product path has no CPU fallback."""
from . import inputs  # noqa: F401

__all__ = ["inputs", "binding", "build"]
