"""B200-native time-sliced tile rasterizer for native 4D Gaussians (arxiv 2412.20720).

``paper_2412_20720_b200.fdgs``   – thin ctypes binding over the C-ABI library (include/fdgs.h)
``paper_2412_20720_b200.scenes`` – seeded synthetic scene / camera generators (no method arithmetic)

Importing the package is cheap; the CUDA library is loaded on the first call into ``fdgs`` and
that call fails loudly if ``libfdgs.so`` has not been built (there is no CPU fallback).
"""
__all__ = ["fdgs", "scenes"]
