"""B200-native SP2 density-matrix hot path of arxiv 2101.06385.

`paper_2101_06385_b200.api` is the thin ctypes binding over the C-ABI library
`libsp2b200.so` (include/sp2_b200.h); `paper_2101_06385_b200.workloads` holds the seeded
synthetic inputs.  Importing the package does not load the CUDA library; the first call
into `api` does, and raises if it is missing (there is no CPU fallback).
"""
__all__ = ["api", "workloads"]
