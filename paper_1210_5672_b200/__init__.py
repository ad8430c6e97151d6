"""paper_1210_5672_b200 -- B200-native Dirichlet-to-Neumann hot path of Wilkening & Yu (arXiv 1210.5672).

Thin Python binding over the C ABI of include/sww.h (libsww.so, hand-written CUDA for sm_100a).  This layer only marshals
arguments: torch supplies device memory and streams, every step of the path runs in the library's kernels.  There is no CPU
fallback: importing works without a GPU (so the build and symbol checks can run), any compute call without CUDA raises.
"""
from .binding import (DtN, State, Shooter, SwwError, lib, lib_path, launch_count, probe_fp64_peak, dtn_linearized_host, host_cache_clear, F64, DD,
                      dd_pack, dd_unpack, EXPORTS, timing_enable, timing_read, KERNEL_CLASSES, lm_minimize, mesh_points, respace_noalloc, RESPACE_NOALLOC_MAX)

__all__ = ["DtN", "State", "Shooter", "SwwError", "lib", "lib_path", "launch_count", "probe_fp64_peak", "dtn_linearized_host", "host_cache_clear", "F64", "DD",
           "dd_pack", "dd_unpack", "EXPORTS", "timing_enable", "timing_read", "KERNEL_CLASSES", "lm_minimize", "mesh_points", "respace_noalloc", "RESPACE_NOALLOC_MAX"]
