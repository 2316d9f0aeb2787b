"""paper_2606_25040_b200 — B200-native hot path of Chorus II's sparsity reuse.

`libchorus.so` (hand-written sm_100a CUDA behind the C ABI in include/chorus.h) plus a thin ctypes
binding with the same names.  Importing the package does not load the library; the first call
does, and fails loudly if it is missing — there is no CPU fallback.
"""
from __future__ import annotations

__all__ = ["binding", "workloads"]
