"""B200-native CSPH-TVD time step (arxiv 1912.04855): CUDA kernels behind a C-ABI.

`workloads` (numpy-only input generators) imports without the CUDA library; the
binding in `cspt` loads `libcspt.so` on first use and fails loudly if it is missing.
"""
__all__ = ["workloads", "cspt"]
