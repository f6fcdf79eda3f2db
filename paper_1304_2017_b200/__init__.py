"""B200-native matched projector pair H / H^T of the interpolation-based D-D
imaging model of 3-D optoacoustic tomography (arxiv/paper_1304_2017, Sec. II.B.1,
II.B.3, III.C, Appendix).

The package holds only what the hot path needs:

  csrc/        CUDA kernels (sm_100a) and the C-ABI library ``liboat.so``
  binding.py   thin ctypes binding with the same names as ``include/oat.h``
  build.py     in-tree nvcc build of ``liboat.so``
  workloads.py seeded synthetic inputs (shared with the oracle's tests; holds
               none of the method's arithmetic)

Importing the package does NOT load the CUDA library; ``binding`` does, and it
fails loudly when the library is missing (there is no CPU fallback).
"""

__all__ = ["binding", "build", "workloads"]
