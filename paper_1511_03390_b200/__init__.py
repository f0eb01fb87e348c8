"""B200-native quadrature lock-in discrimination (QLD) hot path, arXiv 1511.03390.

Importing the package loads nothing native.  `paper_1511_03390_b200.qld` is the thin binding over
the C-ABI library (include/qld.h); it raises if the CUDA library has not been built.
`paper_1511_03390_b200.synth` is the seeded synthetic input generator (numpy only).
"""
__all__ = ["synth", "qld", "build"]
