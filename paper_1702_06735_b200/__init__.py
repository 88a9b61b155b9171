"""tddp4 on B200: time-dependent four-body amplitude likelihood (arXiv:1702.06735) behind a C-ABI.

Importing the package is cheap and never touches CUDA.  `paper_1702_06735_b200.binding` loads the
C-ABI library (csrc/libtddp4.so) and fails loudly if it is missing; there is no CPU fallback.
"""
__all__ = ["workloads", "binding"]
