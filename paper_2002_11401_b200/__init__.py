"""flatspin hot path, B200-native: C-ABI CUDA library (csrc/flatspin.cu, include/flatspin.h) plus a
thin ctypes binding.  `workloads` holds the seeded synthetic input generators.  torch is imported
lazily by `binding` so that the generators can be used without it."""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding", "build"]
