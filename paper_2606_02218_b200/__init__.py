"""B200-native (sm_100a) synchronous group rollout + group-relative advantages.

The product is the C-ABI library `libsagc.so` (include/sagc.h); `binding` is a thin ctypes
layer with the same call names (argument marshalling only).  `workloads` holds the seeded
synthetic input generators.  There is no CPU fallback: importing `binding` without the built
library, or calling it without a CUDA device, fails loudly.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads"]
