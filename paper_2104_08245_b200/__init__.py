"""B200-native NOLSM hot path (arXiv 2104.08245): thin Python binding over the C ABI of
include/nolsm.h.  Argument marshalling only -- every step of the path runs in libnolsm's CUDA kernels.
There is no CPU fallback: without the built library or without a CUDA device the calls raise."""
from .binding import (Context, Config, BlockSparse, Batch, SignStats, SolveStats, NolsmError, load_library, combine_submatrices, union_pattern, Groups,
                      FP16_FP32, FP32, MAT_S, MAT_H, MAT_SINV, MAT_B, MAT_X, FLAG_SIMT_ONLY, FLAG_PAIR, FLAG_SINGLE, FLAG_UNIT_SCALE, FLAG_ORDER3, FLAG_NO_PREDICT, FLAG_LOWDIN, FLAG_NO_RESCALE,
                      EXPORTED_SYMBOLS, library_path)

__all__ = ["Context", "Config", "BlockSparse", "Batch", "SignStats", "SolveStats", "NolsmError", "load_library", "combine_submatrices", "union_pattern", "Groups",
           "FP16_FP32", "FP32", "MAT_S", "MAT_H", "MAT_SINV", "MAT_B", "MAT_X", "FLAG_SIMT_ONLY", "FLAG_PAIR", "FLAG_SINGLE", "FLAG_UNIT_SCALE", "FLAG_ORDER3", "FLAG_NO_PREDICT", "FLAG_LOWDIN", "FLAG_NO_RESCALE",
           "EXPORTED_SYMBOLS", "library_path"]
