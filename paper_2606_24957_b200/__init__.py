"""B200-native sparse verification attention of "Dustin" (arxiv/paper_2606_24957).

The product is the C-ABI library built from csrc/ (include/dustin.h); `paper_2606_24957_b200.api` is the thin
ctypes binding with the same entry-point names.  Importing this package loads nothing: the shared library is
opened on first use and a missing library is a hard error (there is no CPU fallback).
`paper_2606_24957_b200.synth` holds the seeded input generators shared with the oracle's tests.
"""
__all__ = ["api", "synth"]
