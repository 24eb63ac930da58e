"""paper_1912_05529_b200 -- B200-native hot path of explicit f-x poststack depth migration.

Thin Python binding over the C-ABI library libpdm.so (include/pdm.h).  Argument marshalling
only: every step of the path (table look-up, FIR extrapolation, depth marching, imaging) runs
in the CUDA kernels under csrc/.  PyTorch is used for device memory and streams.
"""
from .binding import (Plan, Plan3D, pdm3_create, SectionTransform, pdm_tf_create, pdm_tf_forward, pdm_tf_destroy, PdmError, load_library, pdm_create, pdm_migrate, pdm_migrate_host, pdm_migrate_shot, pdm_migrate_static, migrate_static,  # noqa: F401
                      pdm_destroy, pdm_get_info, pdm_strerror, pdm_debug_table_index,
                      pdm_fp32_peak, pdm_design_table, pdm_profile_enable, pdm_profile_read, PdmInfo, EXPORTED_SYMBOLS,
                      PDM_PATH_AUTO, PDM_PATH_SMEM, PDM_PATH_TILED, PDM_PATH_NAIVE, PDM_PATH_CLUSTER, PDM_PATH_PACKED,
                      PDM_FORCE_GENERAL, PDM_NO_BALANCE, PDM_REQUIRE_SYMMETRIC, PDM_PRESTACK, PDM_TABLE_INTERP, PDM_THREADS_SHIFT, PDM_CTAS_SHIFT, PDM_TAPER_SHIFT,
                      PDM_TAPS_AUTO, PDM_TAPS_GLOBAL, PDM_TAPS_SLICE, PDM_TAPS_COMPACT,
                      PDM_OK, PDM_ERR_INVALID_ARG, PDM_ERR_TABLE_RANGE, PDM_ERR_TABLE_ASYMMETRIC,
                      PDM_ERR_UNSUPPORTED, PDM_ERR_NOMEM, PDM_ERR_CUDA, PDM_ERR_TOO_LARGE, PDM_STATIC_MAX_SAMPLES)
from .build import build_lib  # noqa: F401
