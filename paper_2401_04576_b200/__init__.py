"""B200-native interval-arithmetic helix vote (hot path of arxiv 2401.04576).

`eventgen` (seeded inputs) imports without CUDA; everything that computes goes through the
C-ABI library `libia_b200.so` via `binding` and fails loudly when that library is missing.
"""
__all__ = ["eventgen", "binding"]
