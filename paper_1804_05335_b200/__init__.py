"""
fdas-b200: B200-native FDAS correlation hot path (arXiv:1804.05335) behind a C ABI.

`paper_1804_05335_b200.fdas` is the thin ctypes binding over `libfdas.so` (argument
marshalling only); `paper_1804_05335_b200.synthetic` holds the seeded input generators.
Nothing here falls back to a CPU implementation: importing `fdas` without the built
CUDA library raises.
"""
__all__ = ["fdas", "synthetic"]
