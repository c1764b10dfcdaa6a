"""mfsdp: owner-local Muon / AdamW optimizer step of MatrixFSDP (arxiv/paper_2607_05895) for B200 (sm_100a).

Thin ctypes binding over libmfsdp.so (C ABI in include/mfsdp.h).  Argument marshalling only: every step of the path
runs in the library's CUDA kernels; PyTorch supplies device memory and streams.  There is no CPU fallback -- if the
library is not built the first call raises, and on a machine without an sm_100 device the step functions raise
MfsdpError(MFSDP_EARCH).
"""
from .binding import (  # noqa: F401
    BF16, F32, ROLE_MATRIX, ROLE_TAIL, POLICY_ROLE_GREEDY, POLICY_SCOPE_GREEDY, POLICY_COST_AWARE, METRIC_NUMEL, METRIC_NS_FLOPS,
    SCALE_MATCH_RMS_ADAMW, SCALE_ORIGINAL, SCALE_NONE, NS_BF16, NS_FP32, STEP_KEEP_O,
    EINVAL, ECAP, ELAYOUT, EARCH, ECUDA, ECACHE, ETOOBIG,
    MfsdpError, Param, Desc, MuonHParams, AdamWHParams, PlanResult,
    lib_path, load, exported_symbols,
    mfsdp_plan, mfsdp_plan_ex, mfsdp_score_plan, mfsdp_reduce_schedule, mfsdp_muon_step_gated, mfsdp_signal_ready, mfsdp_muon_step_fanout,
    ReduceOp, Caps, RankScore, BlockScore, mfsdp_validate_desc, mfsdp_flat_elems, mfsdp_workspace_bytes, mfsdp_host_workspace_bytes, mfsdp_workspace_view,
    mfsdp_debug_ws_offsets, mfsdp_muon_step, mfsdp_muon_momentum_pass, mfsdp_muon_ns_pass, mfsdp_muon_update_pass,
    mfsdp_muon_step_host, mfsdp_adamw_tail_step, mfsdp_strerror, mfsdp_version, mfsdp_launch_count,
    mfsdp_tune, mfsdp_get_tune, mfsdp_debug_trace, TUNE_PAIR_MIN_D, TUNE_SYM_BAND, TUNE_SYM_BAND2, TUNE_RECT_GROUP, TUNE_WIDE_MIN_KB, TUNE_FUSED_BELOW_D, TUNE_FUSED2_BELOW_D, mfsdp_release_plans, mfsdp_ns_class,
    make_desc_array, SHAMPOO_KEEP_D, ShampooHParams, mfsdp_shampoo_state_bytes, mfsdp_shampoo_workspace_bytes,
    mfsdp_shampoo_view, mfsdp_shampoo_step, mfsdp_momentum_pass_static, mfsdp_static_max_elems,
)
