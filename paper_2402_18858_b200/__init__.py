"""B200-native ANN chemistry step (arXiv 2402.18858 hot path): C-ABI library + thin ctypes binding.

`inputs` (seeded generators) imports nothing native; `binding` loads libgpuann.so and fails loudly if
it is missing -- there is no CPU fallback.
"""
__all__ = ["inputs", "binding", "build"]
