"""SubQuad candidate-pair affinity path (arxiv/paper_2602_17330), B200-native.

`paper_2602_17330_b200.binding` is the thin Python layer over the C-ABI library
(`include/subquad.h`); `paper_2602_17330_b200.datagen` draws the seeded synthetic
inputs.  Importing the package itself loads neither torch nor the CUDA library.
"""
__all__ = ["binding", "datagen", "build"]
