"""B200-native matched-filter hot path of cuInspiral (arXiv 1006.4644).

`paper_1006_4644_b200.cbmf`      -- thin ctypes binding of the C-ABI library (include/cbmf.h)
`paper_1006_4644_b200.sharding`  -- bank slicing for one process per GPU (index bookkeeping only)

Importing the package does not load the CUDA library; `cbmf` does, and fails
loudly if it is missing (there is no CPU fallback).
"""
__all__ = ["cbmf", "sharding"]
