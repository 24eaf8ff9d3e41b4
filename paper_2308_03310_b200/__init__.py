"""B200-native LETKF local analysis (arXiv 2308.03310): batched fp64 symmetric EVD and the
fused per-grid-point analysis, as hand-written sm_100a CUDA behind a C ABI (include/letkf.h).

The binding is loaded lazily: importing the package does not need
the CUDA extension, but the first call into the hot path does and fails loudly without it.
There is no CPU fallback.
"""

__all__ = ["letkf", "sharding"]
