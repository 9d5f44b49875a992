"""B200-native block-level DDM / WaveHoltz Helmholtz sweep (arxiv/paper_2606_21695).

`paper_2606_21695_b200.hz` is the thin ctypes binding over the C-ABI library declared in
include/hz.h; `paper_2606_21695_b200.inputs` builds the seeded synthetic configs.  Importing
the package does not load the CUDA library; the first call into `hz` does, and raises if the
library has not been built (there is no CPU fallback).
"""
__all__ = ["inputs", "hz"]
