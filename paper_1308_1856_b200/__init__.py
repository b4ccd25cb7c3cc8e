"""B200-native TDSE hot path (CLTDSE method, arXiv:1308.1856): C-ABI CUDA library + thin binding.

Importing the package does not load the CUDA library; `paper_1308_1856_b200.binding` does, and
fails loudly if it is missing (there is no CPU fallback).
"""
__all__ = ["binding", "workloads", "build"]
