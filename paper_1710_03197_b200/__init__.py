"""paper_1710_03197_b200 -- B200-native NUFFT hot path (arxiv 1710.03197, PyNUFFT): A = V F S, A^H, A^H A,
multi-coil operator, CG and L1TV-OLS drivers, as hand-written sm_100a CUDA kernels behind a C ABI
(include/nufft.h).  This package is the thin Python binding: argument marshalling only.

There is no CPU fallback: importing works without a GPU (so that the library's exported symbols can be checked),
but every compute call needs CUDA tensors and raises otherwise.
"""
from .binding import (NufftError, NufftPlan, lib, lib_path, version, EXPORTED_SYMBOLS)  # noqa: F401

__all__ = ["NufftError", "NufftPlan", "lib", "lib_path", "version", "EXPORTED_SYMBOLS"]
