"""tfs: B200-native batch evaluator of the LISA semi-coherent TF statistic Upsilon_Nseg.

``synth`` (seeded inputs) imports without the CUDA library; everything in ``api`` needs
``libtfs.so`` and fails loudly if it is missing (there is no CPU fallback).
"""
__all__ = ["synth", "api"]
