"""paper_2408_01361_b200 -- B200-native hot path of the KHARMA/HARM method (arxiv 2408.01361):
one explicit second-order ideal-GRMHD update of a uniform 3-D block in a stationary metric, fp64,
in hand-written CUDA kernels for sm_100a behind the C ABI of include/kharm.h.

This package is the thin Python binding (argument marshalling only).  There is no CPU fallback:
importing works anywhere, but creating a Grid needs libkharm.so and a CUDA device.
"""
from .binding import (Grid, KharmError, Params, lib, make_params, measure_fp64_peak,  # noqa: F401
                      link_blocks, exchange_halos, step_blocks, divB_noalloc, NOALLOC_MAX_CORNERS,
                      MINKOWSKI, KS, FMKS, BC_PERIODIC, BC_OUTFLOW, BC_POLAR, BC_FIXED, BC_BLOCK, RECON_MC, RECON_WENO5,
                      LOC_CENT, LOC_FACE1, LOC_FACE2, LOC_FACE3, NG, EXPORTED_SYMBOLS, KERNEL_KINDS)
