"""B200-native ECHO RMHD time step (arXiv:2401.03008): C-ABI CUDA library + thin ctypes binding.

`inputs` holds the seeded synthetic workloads; `binding` loads libecho_b200.so and fails loudly
when it is missing (there is no CPU fallback).
"""
__all__ = ["inputs", "binding"]
