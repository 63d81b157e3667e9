"""B200-native multi-RHS Wilson-clover Dslash and batched mixed-precision CG (hot path of arxiv 2510.26313).

`inputs` (seeded synthetic workloads) imports nothing else; `binding` is the ctypes front end of the CUDA
library behind include/lqcd_b200.h and fails loudly if the library is not built.
"""
__all__ = ["inputs", "binding", "build"]
