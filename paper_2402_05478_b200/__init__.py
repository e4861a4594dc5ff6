"""B200-native pseudo-spectral isothermal MHD step (arxiv 2402.05478 hot path).

The product is the C-ABI CUDA library `libmhd_b200.so` (include/mhd.h); `mhd` is its thin ctypes
binding (argument marshalling only) and `inputs` holds the seeded synthetic initial conditions.
"""
__all__ = ["inputs", "mhd", "build"]
