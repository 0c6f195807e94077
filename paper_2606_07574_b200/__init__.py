"""B200-native batched 4x4 Birkhoff (KL / entropic-OT) projection -- arXiv 2606.07574.

The product is the C-ABI library `libbirkhoff4.so` (include/birkhoff4.h, csrc/*.cu, sm_100a); this
package is a thin ctypes binding with the same entry-point names (`binding.py`), the nvcc build step
(`build.py`) and the seeded workload generators (`inputs.py`).  There is no CPU fallback: every
compute call raises if the CUDA library is missing.
"""
__all__ = ["inputs", "binding", "build"]
