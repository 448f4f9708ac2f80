"""B200-native X-engine for the O(N^2) hot path of arXiv 1503.06203 (thin Python binding).

Every step of the path runs in the CUDA kernels behind the C ABI of include/corr.h
(libcorr_b200.so); this package only marshals arguments.  PyTorch is used for device memory
and streams, nothing else.  There is no CPU fallback: if the library is missing or there is no
sm_100 device, calls raise.
"""
from .binding import (CorrError, Plan, PATH_AUTO, PATH_DP4A, PATH_TCGEN05, PATH_IMMA, baseline_index, count_tiles, schedule_pairs,
                      corr_execute, corr_execute_gated, corr_submit_host, corr_wait_host, corr_measure_int8_tops, corr_plan_create, corr_plan_destroy, corr_time_shift, lib_path, load_library,
                      time_shift, corr_execute_noalloc, execute_noalloc, NOALLOC_MAX_BYTES)

__all__ = ["CorrError", "Plan", "PATH_AUTO", "PATH_DP4A", "PATH_TCGEN05", "PATH_IMMA", "baseline_index", "count_tiles", "schedule_pairs",
           "corr_execute", "corr_execute_gated", "corr_submit_host", "corr_wait_host", "corr_measure_int8_tops", "corr_plan_create", "corr_plan_destroy", "corr_time_shift", "lib_path", "load_library",
           "time_shift", "corr_execute_noalloc", "execute_noalloc", "NOALLOC_MAX_BYTES"]
