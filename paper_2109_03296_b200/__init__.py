"""B200-native KBMOD shift-and-stack search hot path (arXiv 2109.03296): Python binding of the C-ABI
library libkbmod_b200.so (include/kbmod_b200.h) plus the seeded synthetic input generators."""
from .binding import (ALGO_AUTO, ALGO_DIRECT, ALGO_PRUNED, KbmodError, Plan, SearchParams,  # noqa: F401
                      kbmod_coadd_stamps, kbmod_coadd_stamps_filtered, kbmod_default_params, kbmod_displacements,
                      kbmod_eval_trajectories, kbmod_measure_smem_gbs, kbmod_pipeline_host,
                      kbmod_pipeline_host_arena_bytes, kbmod_pipeline_host_arena_bytes_for, kbmod_pipeline_host_batch,
                      kbmod_plan_stats, kbmod_prepare_psi_phi, kbmod_release_thread_state, kbmod_search,
                      kbmod_search_phase_ms, kbmod_search_phase_timing, kbmod_search_stats,
                      kbmod_search_unfiltered_lh, kbmod_search_workspace_bytes, kbmod_search_workspace_bytes_for,
                      kbmod_sigmag_filter, kbmod_sigmag_postfilter, kbmod_stamp_moments, kbmod_version)
