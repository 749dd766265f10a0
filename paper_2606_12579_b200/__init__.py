"""B200-native (sm_100a) G-MAPP multi-agent vector-field rollout: C-ABI CUDA library + thin binding.

Importing the package does not load the CUDA library; `paper_2606_12579_b200.api` does, lazily,
and fails loudly if `libgmapp.so` is missing (there is no CPU fallback).
"""
__all__ = ["scenes", "api"]
