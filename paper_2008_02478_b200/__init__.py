"""B200-native demagnetizing-field convolution (hot path of arXiv 2008.02478, Boris).

``workloads`` (seeded synthetic inputs) imports without the CUDA library;
everything that computes goes through ``binding`` -> ``libborisdemag.so`` and
fails loudly if that library is missing.  There is no CPU fallback.
"""
__all__ = ["workloads", "binding"]
