"""B200-native LASP-Adam fitting hot path (arXiv 2512.24840): C-ABI CUDA library + thin binding.

`synth` (seeded input generators) imports without the CUDA library; everything in `binding`
loads `liblasp_gpu.so` and raises loudly when it is missing -- there is no CPU fallback.
"""
__all__ = ["synth", "binding"]
