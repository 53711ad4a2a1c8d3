"""cc-b200: convex clustering (proximal distance MM, arXiv 1409.2065) hot path on NVIDIA B200.

Importing the package does not load the CUDA library; `paper_1409_2065_b200.binding` does, and it
fails loudly when `libcc_b200.so` is missing (there is no CPU fallback).
"""
__all__ = ["synth", "binding"]
