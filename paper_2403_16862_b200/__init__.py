"""B200-native differentiable bilinear point rasterizer (INPC, arXiv 2403.16862, Sec. 3.4 / App. A.6).

`workloads` (seeded synthetic inputs) imports without CUDA; `raster` (the binding over the C-ABI
library built from csrc/) is imported lazily and fails loudly when the library is missing.
"""
__all__ = ["workloads", "raster"]
