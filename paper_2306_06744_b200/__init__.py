"""B200-native linear quadtree/octree h-adaptation hot path (arxiv 2306.06744).

``paper_2306_06744_b200.lt``        thin ctypes binding over the C-ABI CUDA library (include/lt.h)
``paper_2306_06744_b200.workloads`` seeded synthetic inputs (shared with the oracle's tests)

Nothing here imports ``oracle/``; the CUDA library is loaded on first use of ``lt`` and
raises if it is missing (there is no CPU fallback).
"""
__all__ = ["lt", "workloads"]
