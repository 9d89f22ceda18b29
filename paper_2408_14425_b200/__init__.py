"""Radiance-cascades formal solution (arxiv 2408.14425), B200-native hot path.

`atmospheres` (seeded synthetic inputs; numpy only) imports without a GPU.  Everything that
computes goes through `binding` -> librc.so (C ABI, include/rc.h) -> sm_100a kernels; there is
no CPU fallback: `binding.load()` raises if the CUDA library is missing.
"""
__all__ = ["atmospheres", "binding"]
