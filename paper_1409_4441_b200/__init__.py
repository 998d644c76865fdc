"""paper_1409_4441_b200 -- B200-native real-space spherical convolution on HEALPix RING maps.

Thin Python binding (argument marshalling only) of the C-ABI library `libsc.so` declared in
include/sc.h.  Every step of the path runs in the library's CUDA kernels; PyTorch is used by callers
for device memory and streams only.  There is no CPU fallback: without the built library or without
a CUDA device the calls raise.
"""
from .api import (Plan, ScError, lib, sc_plan_create, sc_plan_create_zoned, sc_convolve, sc_convolve_host,  # noqa: F401
                  sc_convolve_profile, sc_plan_partition, KERNEL_NAMES, sc_band_partition, sc_convolve_band, sc_cap_rows, sc_convolve_cap,
                  sc_plan_destroy, sc_plan_info, sc_plan_set_path, sc_debug_neighbour_counts, sc_neighbour_counts_static, SC_STATIC_MAX_NPIX,
                  sc_debug_stats, sc_debug_fma_peak, sc_last_launch_count, sc_plan_double_coordinate, sc_version, EXPORTS,
                  SC_ORDER_RING, SC_ORDER_NESTED, SC_PATH_AUTO, SC_PATH_GENERIC)
