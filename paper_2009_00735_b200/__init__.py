"""paper_2009_00735_b200 -- B200-native signatures for atom-probe crystallography (arXiv 2009.00735).

The product is the CUDA library `libaptsig.so` (sources in csrc/, ABI in include/aptsig.h); this
package is its ctypes binding.  Importing the package does not load the library; the first call does,
and raises if it has not been built (there is no CPU fallback).
"""
from .binding import (Plan, Indexer, apx_so3_grid_cubic, apx_fsp_noalloc_limits, EXT_EXPORTS, APX_INDEX_MAX_K, ApxError, apx_peak_name, apx_peak_measure, PEAK_EXPORTS, apx_dirs_fibonacci, apx_dirs_geodesic, apx_dirs_antipodes, apx_version, EXPORTS, LIB_PATH,
                      APX_FLAG_FORCE_FFT, APX_FLAG_FORCE_MMA, APX_FLAG_NO_PAIRING, APX_FLAG_NORMALISE, APX_FLAG_LOCAL_MAX,
                      APX_PEAK_MAX, APX_PEAK_LOCAL_MAX, APX_MAX_SIGNATURES, APX_OK, APX_EINVAL, APX_ENOMEM, APX_ECUDA,
                      APX_ESTATE, APX_ERANGE)

from .parallel import shard_range, run_sharded, gather_counts
from .refine import adaptive_scan

__all__ = ["Indexer", "apx_so3_grid_cubic", "apx_fsp_noalloc_limits", "EXT_EXPORTS", "APX_INDEX_MAX_K", "adaptive_scan", "apx_peak_name", "apx_peak_measure", "PEAK_EXPORTS", "shard_range", "run_sharded", "gather_counts", "Plan", "ApxError", "apx_dirs_fibonacci", "apx_dirs_geodesic", "apx_dirs_antipodes", "apx_version", "EXPORTS", "LIB_PATH",
           "APX_FLAG_FORCE_FFT", "APX_FLAG_FORCE_MMA", "APX_FLAG_NO_PAIRING", "APX_FLAG_NORMALISE", "APX_FLAG_LOCAL_MAX",
           "APX_PEAK_MAX", "APX_PEAK_LOCAL_MAX", "APX_MAX_SIGNATURES"]
