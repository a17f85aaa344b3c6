"""B200-native batched rigid-body operators (FK, Jacobian, RNEA, CRBA) -- hot path of BARD (arxiv 2605.31481).

Importing the package is cheap and never touches CUDA; ``paper_2605_31481_b200.binding`` loads the C-ABI
library ``libbard.so`` (see ``include/bard.h``) on first use and fails loudly if it is missing.
"""
__all__ = ["workloads"]
