"""B200-native (sm_100a) hot path of the multispecies particle Landau scheme (arXiv:2212.00663).

`workloads` (seeded synthetic inputs) and `analytic` (comparison curves) are plain numpy and load
no native code.  The CUDA path lives behind the C ABI of include/landau.h; `binding` marshals
arguments to it and fails loudly when liblandau.so is missing (there is no CPU fallback).
"""
__all__ = ["workloads", "analytic", "binding", "build"]
