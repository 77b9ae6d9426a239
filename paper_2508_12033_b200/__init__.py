"""B200-native load-balanced LRDMC hot path (arxiv 2508.12033): CUDA kernels behind a C-ABI.

`paper_2508_12033_b200.workloads` (numpy only) is importable everywhere; the binding
(`paper_2508_12033_b200.binding`) loads `liblrdmc.so` lazily and fails loudly if it is missing.
"""
