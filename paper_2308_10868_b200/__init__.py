"""B200-native block matching for physics-based non-rigid registration (arxiv/paper_2308_10868).

The product is libnrr_bm.so (C ABI in include/nrr_bm.h, CUDA kernels in csrc/); this package is its thin
Python binding.  Same names as the C entry points.
"""
from .binding import (  # noqa: F401
    EXPORTS, LIB_PATH, NrrError, lib,
    nrr_bm_check_async_error, nrr_bm_fp32_peak, nrr_bm_fp32_microbench, nrr_bm_launch_count, nrr_bm_match, nrr_bm_register, nrr_bm_moving_stats, nrr_bm_match_host,
    nrr_bm_match_info, nrr_bm_pair_task_table, nrr_bm_profile_enable, nrr_bm_profile_read, nrr_bm_register_host, nrr_bm_select_blocks,
    nrr_bm_select_blocks_pruned,
    nrr_bm_select_blocks_host, nrr_bm_set_option, nrr_bm_version, nrr_bm_warp,
    NrrPlan, nrr_bm_capacity_bound, nrr_bm_plan_blocks, nrr_bm_plan_blocks_host, nrr_bm_plan_create, nrr_bm_plan_create_host, nrr_bm_plan_destroy,
    NrrFem, nrr_bm_fem_create, nrr_bm_fem_dense_field, nrr_bm_fem_dense_field_host, nrr_bm_fem_destroy, nrr_bm_fem_solve,
    nrr_bm_fem_solve_host,
    nrr_bm_plan_info, nrr_bm_plan_match, nrr_bm_plan_match_host, nrr_bm_plan_match_range, nrr_bm_register_batch, nrr_bm_setting,
)
