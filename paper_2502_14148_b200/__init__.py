"""paper_2502_14148_b200 — B200-native (sm_100a) C-grid tendency + RK3 hot path of arXiv 2502.14148.

The product is the C-ABI library `libocn.so` (include/ocn.h, csrc/); `binding` is the thin ctypes
layer with the same call names.  Importing this package loads nothing native; `binding.lib()`
loads the CUDA library and fails loudly if it is missing — there is no CPU fallback.
`workloads` only generates seeded synthetic inputs (used by tests, bench.py and the oracle side).
"""
__all__ = ["binding", "workloads", "build"]
