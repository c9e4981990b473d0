"""B200-native (sm_100a) multiresolution 4D hash encoder of DASH (arxiv 2507.19141, §4.2).

Thin Python binding over the C-ABI library `libdash_hash4d.so` (include/dash_hash4d.h):
argument marshalling only — every step of the path runs in the library's CUDA kernels.
There is no CPU fallback: without the built library or without a CUDA device the calls raise.
"""
from .binding import (  # noqa: F401
    Hash4DConfig, Hash4DError, FLAG_DENSE_COARSE, FLAG_DETERMINISTIC_BWD, FLAG_VALIDATE_INPUTS,
    FLAG_ZERO_GRAD, FLAG_SORT_COARSE, FLAG_ORDER_READY, OP_FWD, OP_BWD, OP_INDICES, OP_BWD_INPUT, OP_SMOOTH, make_config, config_from_params, library_path,
    dash_hash4d_resolutions, dash_hash4d_workspace_bytes, dash_hash3d_workspace_bytes, dash_hash4d_fwd, dash_hash4d_bwd, dash_hash4d_bwd_input, dash_hash4d_smooth,
    dash_hash4d_indices, dash_hash4d_zero, dash_hash4d_last_error, dash_hash4d_launch_count,
    dash_hash3d_resolutions, dash_hash3d_fwd, dash_hash3d_bwd, dash_hash3d_indices, dash_hash3d_bwd_input,
    dash_hash4d_slice_t, dash_hash4d_slice_fwd, dash_deform_slice_fwd, dash_deform_slice_workspace_bytes,
    AdamConfig, ADAM_ZERO_GRAD, dash_hash4d_adam_step,
    MlpConfig, make_mlp_config, dash_mlp_param_count, dash_mlp_fwd, dash_mlp_bwd, dash_deform_bwd, dash_deform_workspace_bytes, dash_deform_fwd,
    dash_hash4d_fwd_host, dash_hash4d_bwd_host, exported_symbols, with_flags, HostStep,
    dash_hash4d_sort_queries, dash_hash4d_sort_queries_static, dash_decompose, dash_decompose_read, DecomposeResult, dash_hash4d_set_debug, DEBUG_FWD_GROUP, DEBUG_BWD_GROUP, DEBUG_SMOOTH_GROUP, DEBUG_DEFORM_PATH,
    DEBUG_BWD_VARIANT, DEBUG_BWD_COARSE_LEVELS, DEBUG_BWD_RUN_CHUNK, DEBUG_FWD_ORDERED_LEVELS, DEBUG_SORT_KEY_BITS,
    dash_ceiling_launch, CEIL_COPY, CEIL_GATHER, CEIL_RED, CEIL_SMEM_ATOMIC, CEIL_TMA_GATHER, CEIL_SMEM_ATOMIC_U64,
    CEIL_INDEPENDENT, CEIL_PAIR_ALIGNED, CEIL_PAIR_XCORNER,
)
