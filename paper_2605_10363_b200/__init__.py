"""kldi — block-filtered Kohn-Sham EXC contractions for B200 (sm_100a), FP64.

The compute path lives in csrc/ (CUDA, C ABI declared in include/kldi.h) and is reached
through `paper_2605_10363_b200.binding`.  Importing this package does not load the shared
library; the first binding call does, and raises if it is missing (no CPU fallback).
"""
__all__ = ["binding", "workloads"]
