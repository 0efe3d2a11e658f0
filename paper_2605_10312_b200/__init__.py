"""B200-native batched HGP electron-repulsion integrals (hot path of arxiv/paper_2605_10312).

`rcg` is the thin binding over the C-ABI library (csrc/); `workloads` holds the seeded
synthetic inputs.  Importing this package does not load the CUDA library; the first call
into `rcg` does, and fails loudly if it is missing (there is no CPU fallback).
"""
__all__ = ["rcg", "workloads"]
