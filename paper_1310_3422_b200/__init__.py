"""paper_1310_3422_b200 -- B200-native time-marching loop of the group-explicit (GE)
finite-difference scheme of arXiv 1310.3422.

  libge.py   thin ctypes binding of the C ABI in include/ge.h (libge.so, CUDA sm_100a)
  build.py   in-tree nvcc build of libge.so
  inputs.py  seeded synthetic inputs for the BASELINE.json configs (no method arithmetic)
  csrc/      the CUDA kernels and the C ABI

Importing the package does not load CUDA; `libge.load()` does and fails loudly
when libge.so is missing -- there is no CPU fallback.
"""
__all__ = ["libge", "inputs", "build"]
