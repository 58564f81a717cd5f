"""B200-native batched ADMM for the Lightning-style radiosurgery LP (arXiv 2509.08602).

The product is `libadmm_b200.so` (C ABI in include/admm_b200.h, CUDA sm_100a kernels in csrc/);
this package is its thin ctypes binding.  Importing `paper_2509_08602_b200.binding` fails loudly
if the library has not been built; nothing here falls back to the CPU.
"""
__all__ = ["binding", "build"]
