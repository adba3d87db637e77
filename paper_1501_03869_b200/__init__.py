"""B200-native phase-corrected back projection (arxiv 1501.03869, Eq. 7).

The product is the C-ABI library built from csrc/ (libpat_b200.so, sm_100a); this package
is a thin ctypes binding with the same entry-point names.  There is no CPU fallback: the
import fails loudly if the library is missing, and every compute call needs a B200.
"""
from .binding import (PAT_OK, PAT_ERR_INVALID_ARG, PAT_ERR_BAD_STATE, PAT_ERR_CUDA, PAT_ERR_NOMEM,
                      PAT_ERR_UNSUPPORTED, PAT_W_DELAY_SUM, PAT_W_PAPER, PAT_W_PAPER_EXACT, PAT_W_UBP, PAT_W_UBP_EXACT, PatError, PatGrid,
                      lib, library_path, pat_plan_workspace_bytes, pat_plan_create,
                      pat_set_travel_times, pat_backproject, pat_destroy, pat_last_error,
                      pat_kernel_launches, pat_chained_calls, pat_set_device_allocator, pat_get_stats, install_torch_allocator,
                      torch_alloc, torch_free, PatStats, pat_set_gather_tuning, pat_fmm_travel_times,
                      pat_compute_travel_times, pat_set_profiling, pat_get_profile,
                      pat_eikonal_travel_times_device, pat_eikonal_last_stats, pat_pixel_order, pat_compute_travel_times_gpu,
                      pat_backproject_conventional, pat_backproject_conventional_sweep, pat_set_roi_mask, pat_set_pixel_weights,
                      pat_compute_solid_angle_weights, pat_get_trace_window, Plan,
                      pat_backproject_static, pat_backproject_static_max_samples, pat_backproject_static_last_error)

__all__ = [n for n in dir() if n.startswith(("pat_", "PAT_", "Pat", "Plan", "lib"))]
