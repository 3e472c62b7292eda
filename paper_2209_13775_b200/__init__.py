"""B200-native hot path of the LCS pipeline of arXiv 2209.13775 (Ameli, Desai, Shadden).

Sub-modules (nothing heavy is imported here so that ``inputs`` can be used on its own):
  inputs  - seeded synthetic workloads (serves the CUDA path and the oracle alike)
  lcs     - ctypes binding of liblcs.so, the C-ABI over the sm_100a kernels
  build   - nvcc build of liblcs.so (in-tree)
"""
__all__ = ["inputs", "lcs", "build"]
