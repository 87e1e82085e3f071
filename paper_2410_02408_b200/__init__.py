"""B200-native block-Jacobi preconditioning path of arxiv 2410.02408.

`binding` is the thin ctypes layer over the C-ABI CUDA library `libbj.so` (include/bj.h);
`workloads` holds the seeded synthetic input generators; `sweep` is the host-side block-size
sweep that stands in for the paper's tuner.  Importing the package does not load the CUDA
library; the first call through `binding` does, and fails loudly if it is missing.
"""
__all__ = ["binding", "workloads", "build", "sweep"]
