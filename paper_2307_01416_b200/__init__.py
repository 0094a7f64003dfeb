"""B200-native VPMC transport-and-scoring path (arXiv 2307.01416): C-ABI library `libvpmc.so` + thin binding.

`workloads` (seeded synthetic inputs, numpy only) imports without a GPU; `binding` loads the CUDA library and
fails loudly when it is missing -- there is no CPU fallback.
"""
__all__ = ["workloads", "binding"]
