"""B200-native modal time-stepping (arXiv 2505.05940 hot path): thin ctypes binding over libmodal.so.

Importing the package does not load the CUDA library; ``paper_2505_05940_b200.binding`` does, and
fails loudly if it is missing (there is no CPU fallback).
"""
__all__ = ["workloads"]
