"""B200-native ETICS hot path (SCF + MEX expansion force calculation), arxiv 1406.4254.

Importing the package is cheap and GPU-free; the CUDA C-ABI library is loaded on first use of
`paper_1406_4254_b200.binding` and fails loudly if it is missing (there is no CPU fallback).
"""
__all__ = ["workloads", "binding", "build"]
