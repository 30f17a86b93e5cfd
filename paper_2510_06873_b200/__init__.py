"""paper_2510_06873_b200 — B200-native per-step metadynamics hot path (GPU-MetaD, arxiv 2510.06873).

Sub-modules:
  inputs   seeded synthetic workloads (shared with the oracle tests; no method arithmetic)
  metad    thin ctypes binding over the C-ABI library csrc/ -> libmetad_b200.so (include/metad.h)
Importing the package loads nothing native; ``metad`` fails loudly if the CUDA library is missing.
"""
__all__ = ["inputs", "metad"]
