"""B200-native KBMOD shift-and-stack search hot path (arXiv 2109.03296): Python binding of the C-ABI
library libkbmod_b200.so (include/kbmod_b200.h) plus the seeded synthetic input generators."""
from .binding import (ALGO_AUTO, ALGO_DIRECT, ALGO_PRUNED, KbmodError, SearchParams, kbmod_coadd_stamps,  # noqa: F401
                      kbmod_default_params, kbmod_measure_smem_gbs, kbmod_displacements, kbmod_eval_trajectories, kbmod_plan_stats, kbmod_pipeline_host, kbmod_pipeline_host_batch,
                      kbmod_pipeline_host_arena_bytes, kbmod_prepare_psi_phi, kbmod_search, kbmod_search_stats, kbmod_search_phase_ms, kbmod_search_phase_timing,
                      kbmod_search_workspace_bytes, kbmod_sigmag_filter, kbmod_stamp_moments, kbmod_version)
