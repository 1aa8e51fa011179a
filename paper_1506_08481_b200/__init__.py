"""B200-native far-field mobility product of Spectral Ewald Accelerated Stokesian Dynamics.

Thin Python binding (argument marshalling only) over the C-ABI library ``libse_mobility.so``
(``include/se_mobility.h``); every step of the path runs in the library's CUDA kernels.  PyTorch is
used for device memory and streams only.  There is no CPU fallback: importing works anywhere, but
creating a plan without the built library or without a CUDA device raises.
"""
from .binding import (SE_NUM_STAGES, SE_OPT_REAL_CTAS, SE_OPT_REAL_OVERLAP, SE_OPT_XY_PATH, SE_OPT_YZ_FUSED, SE_OPT_GRAPH, SE_OPT_PAIR_CACHE, SE_OPT_SIZE_VARIANT, SE_OPT_GRID_FP32, SE_VARIANT_HYBRID, SE_VARIANT_REAL, SE_VARIANT_WAVE, SE_SKIP_ONEBODY, SE_SKIP_REAL, SE_SKIP_SELF, SE_SKIP_WAVE, SE_TIMING, SE_CUFFT3D,
                      STAGE_NAMES, SeError, SePlan, declared_symbols, load_library, measure_fp64_peak,
                      version, real_noalloc, SE_NOALLOC_MAX_N)

__all__ = ["SePlan", "SeError", "load_library", "declared_symbols", "version", "measure_fp64_peak", "SE_SKIP_REAL", "SE_SKIP_WAVE",
           "SE_SKIP_SELF", "SE_SKIP_ONEBODY", "SE_TIMING", "SE_CUFFT3D", "SE_NUM_STAGES", "STAGE_NAMES",
           "SE_OPT_REAL_OVERLAP", "SE_OPT_REAL_CTAS", "SE_OPT_XY_PATH", "SE_OPT_YZ_FUSED", "SE_OPT_GRAPH", "SE_OPT_PAIR_CACHE", "SE_OPT_SIZE_VARIANT", "SE_OPT_GRID_FP32",
           "SE_VARIANT_HYBRID", "SE_VARIANT_REAL", "SE_VARIANT_WAVE", "real_noalloc", "SE_NOALLOC_MAX_N"]
