"""B200-native per-cell thermochemistry update of arXiv 2312.05800.

Importing the package is cheap; the CUDA C-ABI library (csrc/ -> libdfthermo.so) is only
loaded when `paper_2312_05800_b200.binding` is used, and that fails loudly if it is missing.
"""
__all__ = ["synth", "binding", "build"]
