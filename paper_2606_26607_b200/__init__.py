"""B200-native Moebius TP<->EP reshard (arXiv 2606.26607): Python binding of the C-ABI library.

Argument marshalling only -- every step of the hot path runs in `libmoebius.so` (host planner in
C++, one persistent sm_100a kernel).  There is no CPU fallback and nothing here imports `oracle/`.
Importing this package fails loudly if the library has not been built
(`python paper_2606_26607_b200/build.py` or `__graft_entry__.build()`).
"""
from ._binding import (  # noqa: F401
    MOEBIUS_TP, MOEBIUS_EP, MOEBIUS_BF16, MOEBIUS_FP32, MOEBIUS_FP8_E4M3_B128,
    T_GATE, T_UP, T_DOWN, T_KPOOL, T_VPOOL, T_GATE_SCALE, T_UP_SCALE, T_DOWN_SCALE,
    T_W13, T_W2, T_W13_SCALE, T_W2_SCALE, T_WQ, T_WK, T_WV, T_WO, ATTN_NONE, ATTN_DUAL, ATTN_GATHER,
    MoebiusError, moebius_config_t, moebius_layout_t, moebius_view_t, moebius_stats_t,
    moebius_create, moebius_destroy, moebius_layout, moebius_view, moebius_bind, moebius_active_mode,
    moebius_plan, moebius_plan_destroy, moebius_block_tables, moebius_plan_stats, moebius_plan_export,
    moebius_reshard, moebius_stage_plan, moebius_reshard_staged, moebius_set_timing, moebius_last_kernel_ms, moebius_kernel_ms_history, moebius_set_launch, moebius_set_tma, moebius_set_ring, moebius_set_l2_policy, moebius_set_kv_rounds, moebius_set_kv_slice, moebius_set_chain_bands, moebius_set_xt_mode,
    moebius_policy_config_t, moebius_policy_preset, moebius_policy_config, moebius_policy_create, moebius_policy_destroy,
    moebius_policy_mode, moebius_policy_step, moebius_capacity_check, moebius_policy_calibrate,
    POLICY_INTERACTIVE, POLICY_ROLLOUT, DECISION_STAY, DECISION_SWITCH, DECISION_CANCELLED,
    moebius_naive_scratch_bytes, moebius_reshard_naive, moebius_static_scratch_bytes, moebius_reshard_naive_static,
    moebius_reshard_shares,
    moebius_share_stats, moebius_plan_waves, moebius_reshard_share, moebius_reshard_publish,
    moebius_arena_create, moebius_arena_destroy, moebius_arena_base, moebius_arena_ready, moebius_arena_export,
    moebius_arena_import,
    moebius_status_str, moebius_version, lib_path, EXPORTED_SYMBOLS, SEG_DTYPE, KV_DTYPE, C2D_DTYPE, BULK_DTYPE,
)
from .session import Session, make_config  # noqa: F401
