"""B200-native hot path of arxiv 1604.03360 (relativistic hydro: L(u) x3 per SSP-RK3 step).

Importing the package does not load the CUDA library; ``paper_1604_03360_b200.binding`` does, and
fails loudly if ``libhydro_b200.so`` has not been built (there is no CPU fallback).
"""
__all__ = ["workloads", "binding"]
