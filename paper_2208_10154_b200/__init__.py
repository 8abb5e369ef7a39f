"""paper_2208_10154_b200 -- B200-native batched spherical harmonic transforms (arXiv:2208.10154 hot path).

`inputs` (NumPy only) is importable anywhere; `binding` loads the CUDA C-ABI library and fails loudly
if it has not been built (there is no CPU fallback).
"""
__all__ = ["inputs", "binding"]
