"""B200-native Chebyshev polynomial filter of ChASE (arXiv 1805.10121, Alg. 4 / Eq. 7).

The product is libchase_filter.so (C ABI: include/chase_filter.h; CUDA sources: csrc/).
This package is its thin Python binding plus the seeded workload generators.
"""
from .binding import (  # noqa: F401
    CHASE_C64, CHASE_C128, CHASE_F32, CHASE_F64, ChaseFilterError,
    chase_degrees, chase_filter, chase_hemm_rows, chase_rows_barrier, chase_rows_signal, chase_rows_wait, chase_rows_status,
    chase_filter_rows_ws,
    chase_ipc_export, chase_ipc_open, chase_ipc_close, chase_lanczos, chase_lanczos_ritz_vectors, chase_lanczos_workspace_bytes, chase_spectral_estimates, chase_filter_host, chase_hemm, chase_residuals,
    chase_residuals_workspace_bytes, chase_filter_kernel_path, chase_filter_launch_count,
    chase_filter_scalars, chase_filter_schedule, chase_filter_step_plan, chase_filter_strerror,
    chase_filter_workspace_bytes, chase_filter_ws, chase_fp64_peak_probe, lib_path, load,
    chase_residuals_static, CHASE_STATIC_SCRATCH_BYTES, chase_scratch_cache_release, HostFilter,
)
