"""B200-native multi-level (FPN) RoIAlign forward + backward (RoIExtractor).

The product is the C-ABI library built from csrc/ (include/raf.h); `binding` is a thin ctypes
marshaller with the same entry-point names.  `inputs` (numpy only) draws the seeded workloads.
Nothing here falls back to a CPU path: calling an op without the built CUDA library raises.
"""
__all__ = ["binding", "inputs", "build"]
