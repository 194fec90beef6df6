"""B200-native hot path of arXiv 2412.12360 (FDTDX): Yee FDTD time stepping and its
time-reversed adjoint as hand-written sm_100a CUDA behind a C ABI (include/fdtd.h).

Importing this package loads no native code; `paper_2412_12360_b200.binding` loads the
shared library (and fails loudly if it is missing -- there is no CPU fallback).
"""
__all__ = ["binding", "workloads", "build"]
