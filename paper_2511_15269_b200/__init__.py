"""B200-native adaptive Laplace FMM evaluate path (arXiv 2511.15269), behind a C-ABI library.

`paper_2511_15269_b200.fmm` is the thin Python binding of include/fmm.h (loads the in-tree CUDA
library and fails loudly if it is missing); `paper_2511_15269_b200.inputs` holds the seeded
synthetic workloads.  Nothing here imports the CPU oracle.
"""
__all__ = ["fmm", "inputs"]
