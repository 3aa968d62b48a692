"""B200-native batched fixed-lag SE(2) SLAM backbone (arxiv/paper_2603_25834, §III-D).

The product is the C-ABI library declared in ``include/slam.h`` (built from ``csrc/``) and the thin
ctypes binding in :mod:`paper_2603_25834_b200.binding`.  Importing this package does NOT load the
CUDA library; ``binding`` does, and fails loudly if it is missing (there is no CPU fallback).

The seeded synthetic-input generator, the roofline work model and the replica helpers are harness code and
live in the top-level ``harness/`` package, not here.
"""

__all__ = ["binding", "build"]
