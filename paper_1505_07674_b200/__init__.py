"""B200-native batched lens likelihood (Lensed, arXiv:1505.07674) -- see DESIGN.md.

`paper_1505_07674_b200.lensed` is the thin Python binding of the C-ABI library
(include/lensed.h); `paper_1505_07674_b200.synth` makes the seeded synthetic inputs.
Nothing is imported eagerly so that the input generator can be used without CUDA.
"""
__all__ = ["lensed", "synth"]
