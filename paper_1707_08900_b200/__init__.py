"""fd6-rk3-b200: B200-native hot path of arXiv 1707.08900 (sixth-order finite-difference
compressible hydrodynamics, 2N-storage RK3).

  paper_1707_08900_b200.fd6     ctypes binding of the C-ABI library (include/fd6.h); importing it
                                loads csrc's libfd6.so and raises if it is missing — there is no
                                CPU fallback anywhere in this package.
  paper_1707_08900_b200.inputs  seeded synthetic inputs (no method arithmetic).
  paper_1707_08900_b200.build   nvcc build of libfd6.so for sm_100a.
  paper_1707_08900_b200.replicas  barrier / max-over-ranks bookkeeping of the "replicas only" multi-GPU mode.
"""
__all__ = ["inputs", "build", "fd6", "replicas"]
