"""fdemri: B200-native frequency-domain EMRI harmonic sum (arXiv:2307.12585), FP64, sm_100a.

The product is the C-ABI CUDA library libfdemri.so (include/fdemri.h); this package is its thin binding
plus the seeded input generator (`synth`).  There is no CPU fallback.
"""
from . import synth  # noqa: F401
from .binding import (FDEMRI_FLAG_BIN_MAJOR, FDEMRI_FLAG_TILE_MAJOR, FDEMRI_FLAG_TIMING, FdemriError, Waveform, fdemri_build_splines, fdemri_destroy, fdemri_get_coeffs,  # noqa: F401
                      fdemri_get_kernel_ms, fdemri_get_item_evals, fdemri_get_stats, fdemri_measure_fp64_peak, fdemri_measure_fp64_peak_3reg, fdemri_measure_issue_ns, fdemri_plan, fdemri_plan_kerr, fdemri_build_splines_kerr, fdemri_select_modes, fdemri_select_modes_rule, fdemri_select_modes_static, FDEMRI_STATIC_MAX_TOTALS, FDEMRI_SELECT_OWN_POWER, FDEMRI_SELECT_CUMULATIVE, fdemri_set_mode_mask, fdemri_set_workspace, fdemri_sum, fdemri_td_sum, fdemri_sum_inner, fdemri_version,
                      fdemri_workspace_bytes, fdemri_workspace_bytes_min, waveform_from_workload)
