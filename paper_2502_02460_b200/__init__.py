"""B200-native reduction of the generalized eigenproblem HC = eps SC to standard form and the
eigenvector back-transform: hand-written sm_100a CUDA kernels behind the C ABI of
`include/gs.h`, plus this thin Python binding.

Importing the package does not load the CUDA library; `paper_2502_02460_b200.gs` does, and fails
loudly if `libgs.so` has not been built (`python -m paper_2502_02460_b200.build`).  There is no CPU
fallback anywhere in this package.
"""

__all__ = ["workloads", "gs", "metrics", "build"]
