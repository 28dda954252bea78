"""B200-native particle-mesh-particle exchange step (arxiv 2509.18261, Sec. 2.2 + Sec. 3).

`inputs` (seeded synthetic workloads) imports without CUDA; `pm` (the thin binding over the C-ABI
library libpm_b200.so) loads the CUDA library on first use and fails loudly if it is missing.
"""
__all__ = ["inputs", "pm"]
