"""B200-native time-sliced tile rasterizer for native 4D Gaussians (arxiv 2412.20720).

``paper_2412_20720_b200.fdgs``   – thin ctypes binding over the C-ABI library (include/fdgs.h)
``paper_2412_20720_b200.scenes`` – seeded synthetic scene / camera generators (no method arithmetic)
``paper_2412_20720_b200.autograd`` – torch.autograd front end (Rasterizer) over the same calls
``paper_2412_20720_b200.sweep``  – secondary measurements (configs 2, 4, 5)

Importing the package is cheap; the CUDA library is loaded on the first call into ``fdgs`` and
that call fails loudly if ``libfdgs.so`` has not been built (there is no CPU fallback).
"""
__all__ = ["fdgs", "scenes", "autograd", "sweep"]
