"""ctypes marshalling for include/moebius.h.  Same names, same semantics; errors raise."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = os.path.join(_HERE, "libmoebius.so")

MOEBIUS_TP, MOEBIUS_EP = 0, 1
MOEBIUS_BF16, MOEBIUS_FP32, MOEBIUS_FP8_E4M3_B128 = 0, 1, 2
T_GATE, T_UP, T_DOWN, T_KPOOL, T_VPOOL, T_GATE_SCALE, T_UP_SCALE, T_DOWN_SCALE = range(8)
T_W13, T_W2, T_W13_SCALE, T_W2_SCALE = range(8, 12)   # w_orient = 1
T_WQ, T_WK, T_WV, T_WO = range(12, 16)                 # attention projections
ATTN_NONE, ATTN_DUAL, ATTN_GATHER = 0, 1, 2

EXPORTED_SYMBOLS = [
    "moebius_create", "moebius_destroy", "moebius_layout", "moebius_view", "moebius_bind",
    "moebius_active_mode", "moebius_plan", "moebius_plan_destroy", "moebius_block_tables",
    "moebius_plan_stats", "moebius_plan_export", "moebius_reshard", "moebius_stage_plan", "moebius_reshard_staged",
    "moebius_naive_scratch_bytes", "moebius_reshard_naive", "moebius_static_scratch_bytes", "moebius_reshard_naive_static",
    "moebius_reshard_shares",
    "moebius_share_stats", "moebius_plan_waves", "moebius_reshard_share", "moebius_reshard_publish",
    "moebius_arena_create", "moebius_arena_destroy", "moebius_arena_base", "moebius_arena_ready",
    "moebius_arena_export", "moebius_arena_import",
    "moebius_set_timing", "moebius_policy_preset", "moebius_policy_create", "moebius_policy_destroy",
    "moebius_policy_mode", "moebius_policy_step", "moebius_capacity_check", "moebius_policy_calibrate",
    "moebius_last_kernel_ms", "moebius_kernel_ms_history", "moebius_set_launch", "moebius_set_tma", "moebius_set_ring", "moebius_set_l2_policy", "moebius_set_kv_rounds", "moebius_set_kv_slice", "moebius_set_chain_bands", "moebius_set_xt_mode", "moebius_status_str", "moebius_version",
]


class MoebiusError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__("%s: %s (%d)" % (where, moebius_status_str(status), status))


class moebius_config_t(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("R", C.c_int32), ("L", C.c_int32), ("E", C.c_int32),
                ("H", C.c_int32), ("I", C.c_int32), ("w_dtype", C.c_int32), ("w_orient", C.c_int32),
                ("kv_heads", C.c_int32), ("head_dim", C.c_int32), ("page_tokens", C.c_int32),
                ("kv_dtype", C.c_int32), ("kv_pool_bytes_per_rank_layer", C.c_int64),
                ("max_requests", C.c_int32), ("max_pages_per_request", C.c_int32),
                ("staging_cap_bytes", C.c_int64), ("n_q_heads", C.c_int32), ("attn_mode", C.c_int32),
                ("w_inplace", C.c_int32), ("reserved0", C.c_int32)]


class moebius_policy_config_t(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("W", C.c_int32), ("T_h", C.c_double), ("T_l", C.c_double),
                ("cooldown_s", C.c_double)]


POLICY_INTERACTIVE, POLICY_ROLLOUT = 0, 1
DECISION_STAY, DECISION_SWITCH, DECISION_CANCELLED = 0, 1, 2


class moebius_layout_t(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("pages_tp", C.c_int32), ("pages_ep", C.c_int32),
                ("tp_page_bytes", C.c_int32), ("ep_page_bytes", C.c_int32), ("base_bytes", C.c_int64),
                ("rank_stride_bytes", C.c_int64), ("weight_slot_bytes", C.c_int64),
                ("weight_spare_bytes", C.c_int64), ("staging_bytes", C.c_int64), ("desc_bytes", C.c_int64),
                ("table_bytes", C.c_int64), ("resident_bytes", C.c_int64), ("tbl_owner_off", C.c_int32),
                ("tbl_lens_off", C.c_int32), ("tbl_bt_off", C.c_int32), ("tbl_reserved", C.c_int32),
                ("attn_full_bytes", C.c_int64), ("attn_dup_bytes", C.c_int64), ("w_staging_bytes", C.c_int64),
                ("w_shift_slots", C.c_int32), ("reserved1", C.c_int32)]


class moebius_view_t(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("ndim", C.c_int32), ("elem_bytes", C.c_int32),
                ("offset", C.c_int64), ("shape", C.c_int64 * 4), ("stride", C.c_int64 * 4)]


class moebius_stats_t(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_segments", C.c_int32), ("n_kv_moves", C.c_int32),
                ("n_kv_rounds", C.c_int32), ("n_kv_staged", C.c_int32), ("n_pool_groups", C.c_int32),
                ("n_units", C.c_int64), ("w_moved", C.c_int64), ("w_relocated", C.c_int64),
                ("w_read", C.c_int64), ("kv_moved", C.c_int64), ("kv_relocated", C.c_int64),
                ("kv_read", C.c_int64), ("staging_used_bytes", C.c_int64),
                ("desc_upload_bytes", C.c_int64), ("table_upload_bytes", C.c_int64),
                ("attn_moved", C.c_int64), ("attn_relocated", C.c_int64), ("attn_read", C.c_int64),
                ("w_staged_bytes", C.c_int64), ("n_w_waves", C.c_int32), ("n_w_parked", C.c_int32)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "struct_size"}


# numpy mirrors of the exported work-list records (diagnostics / hazard tests)
SEG_DTYPE = np.dtype([
    ("kind", "<u4"), ("ep_is_src", "<u4"), ("wait_ctr", "<i4"), ("wait_target", "<u4"),
    ("signal_ctr", "<i4"), ("unit_begin", "<u4"), ("n_units", "<u4"), ("run_bytes", "<u4"),
    ("n_groups", "<u4"), ("rep", "<u4"), ("rows_per_unit", "<u4"), ("groups_per_unit", "<u4"),
    ("chunk_bytes", "<u4"), ("chunks_per_run", "<u4"), ("rows_total", "<u4"), ("row_blocks", "<u4"),
    ("ep_off", "<i8"), ("tp_off", "<i8"), ("kv_mode", "<u4"), ("desc_begin", "<u4"), ("n_desc", "<u4"),
    ("pool_begin", "<u4"), ("n_pools", "<u4"), ("pools_per_unit", "<u4"), ("ep_page_bytes", "<u4"),
    ("tp_page_bytes", "<u4"), ("pool_bytes", "<i8"), ("stg_pool_begin", "<u4"), ("stg_pools", "<u4")])
KV_DTYPE = np.dtype([("ep_rank", "<i4"), ("ep_page", "<i4"), ("tp_page", "<i4"), ("ntok_slot", "<u4")])
C2D_DTYPE = np.dtype([("src_off", "<i8"), ("dst_off", "<i8"), ("rows", "<u4"), ("run_bytes", "<u4"),
                      ("src_stride", "<u4"), ("dst_stride", "<u4")])
BULK_DTYPE = np.dtype([("src_off", "<i8"), ("dst_off", "<i8")])
WBLK_DTYPE = np.dtype([("q", "<u4"), ("row0", "<u4"), ("nrows", "<u4"), ("slot", "<u4")])
assert SEG_DTYPE.itemsize == 128 and KV_DTYPE.itemsize == 16 and C2D_DTYPE.itemsize == 32 and BULK_DTYPE.itemsize == 16


def lib_path() -> str:
    return _LIB


if not os.path.exists(_LIB):
    raise ImportError(
        "libmoebius.so is not built (%s). Build it with `python paper_2606_26607_b200/build.py` "
        "(nvcc, sm_100a). There is no CPU fallback." % _LIB)
_lib = C.CDLL(_LIB)

_vp = C.c_void_p
_i32p = C.POINTER(C.c_int32)
_lib.moebius_create.argtypes = [C.POINTER(moebius_config_t), C.POINTER(_vp)]
_lib.moebius_destroy.argtypes = [_vp]
_lib.moebius_destroy.restype = None
_lib.moebius_layout.argtypes = [_vp, C.POINTER(moebius_layout_t)]
_lib.moebius_view.argtypes = [_vp, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(moebius_view_t)]
_lib.moebius_bind.argtypes = [_vp, _vp, _vp, _vp, _vp, C.c_int]
_lib.moebius_active_mode.argtypes = [_vp]
_lib.moebius_plan.argtypes = [_vp, C.c_int, C.c_int, C.c_int32, _vp, _vp, _vp, C.POINTER(_vp)]
_lib.moebius_plan_destroy.argtypes = [_vp]
_lib.moebius_plan_destroy.restype = None
_lib.moebius_block_tables.argtypes = [_vp, _vp, _vp]
_lib.moebius_plan_stats.argtypes = [_vp, C.POINTER(moebius_stats_t)]
_lib.moebius_plan_export.argtypes = [_vp, C.c_int, _vp, C.c_int64, C.POINTER(C.c_int64)]
_lib.moebius_reshard.argtypes = [_vp, _vp, _vp]
_lib.moebius_policy_preset.argtypes = [C.c_int, C.c_double, C.c_double, C.POINTER(moebius_policy_config_t)]
_lib.moebius_policy_create.argtypes = [C.POINTER(moebius_policy_config_t), C.c_int, C.POINTER(_vp)]
_lib.moebius_policy_destroy.argtypes = [_vp]
_lib.moebius_policy_destroy.restype = None
_lib.moebius_policy_mode.argtypes = [_vp]
_lib.moebius_policy_step.argtypes = [_vp, _vp, C.c_double, C.c_int32, _vp, _i32p, _i32p]
_lib.moebius_capacity_check.argtypes = [_vp, C.c_int, C.c_int32, _vp]
_lib.moebius_policy_calibrate.argtypes = [C.c_int32, _vp, _vp, _vp, _i32p]
_lib.moebius_plan_waves.argtypes = [_vp, _i32p]
_lib.moebius_share_stats.argtypes = [_vp, C.c_int, C.c_int, C.c_int, _vp]
_lib.moebius_reshard_share.argtypes = [_vp, _vp, C.c_int, C.c_int, C.c_int, _vp]
_lib.moebius_reshard_publish.argtypes = [_vp, _vp, _vp]
_lib.moebius_arena_create.argtypes = [_vp, C.c_int, C.c_int, C.c_int, C.POINTER(_vp)]
_lib.moebius_arena_destroy.argtypes = [_vp]
_lib.moebius_arena_destroy.restype = None
_lib.moebius_arena_base.argtypes = [_vp]
_lib.moebius_arena_base.restype = _vp
_lib.moebius_arena_ready.argtypes = [_vp]
_lib.moebius_arena_export.argtypes = [_vp, C.c_int, _i32p]
_lib.moebius_arena_import.argtypes = [_vp, C.c_int, C.c_int]
_lib.moebius_stage_plan.argtypes = [_vp, _vp]
_lib.moebius_reshard_staged.argtypes = [_vp, _vp]
_lib.moebius_set_timing.argtypes = [_vp, C.c_int]
_lib.moebius_last_kernel_ms.argtypes = [_vp, C.POINTER(C.c_float)]
_lib.moebius_kernel_ms_history.argtypes = [_vp, C.POINTER(C.c_float), C.c_int, C.POINTER(C.c_int)]
_lib.moebius_set_launch.argtypes = [_vp, C.c_int, C.c_int, C.c_int]
_lib.moebius_set_tma.argtypes = [_vp, C.c_int, C.c_int, C.c_int]
_lib.moebius_set_ring.argtypes = [_vp, C.c_int, C.c_int]
_lib.moebius_set_l2_policy.argtypes = [_vp, C.c_int, C.c_int]
_lib.moebius_set_kv_rounds.argtypes = [_vp, C.c_int]
_lib.moebius_status_str.argtypes = [C.c_int]
_lib.moebius_status_str.restype = C.c_char_p
_lib.moebius_version.restype = C.c_int


def moebius_status_str(status: int) -> str:
    return _lib.moebius_status_str(int(status)).decode()


def moebius_version() -> int:
    return _lib.moebius_version()


def _chk(status: int, where: str):
    if status != 0:
        raise MoebiusError(status, where)


def moebius_create(cfg: moebius_config_t):
    cfg.struct_size = C.sizeof(moebius_config_t)
    out = _vp()
    _chk(_lib.moebius_create(C.byref(cfg), C.byref(out)), "moebius_create")
    return out


def moebius_destroy(ctx):
    _lib.moebius_destroy(ctx)


def moebius_layout(ctx) -> moebius_layout_t:
    out = moebius_layout_t()
    out.struct_size = C.sizeof(moebius_layout_t)
    _chk(_lib.moebius_layout(ctx, C.byref(out)), "moebius_layout")
    return out


def moebius_view(ctx, mode: int, rank: int, layer: int, tensor_id: int) -> moebius_view_t:
    out = moebius_view_t()
    out.struct_size = C.sizeof(moebius_view_t)
    _chk(_lib.moebius_view(ctx, mode, rank, layer, tensor_id, C.byref(out)), "moebius_view")
    return out


def moebius_bind(ctx, dev_base: int, dev_staging: int, dev_desc: int, dev_tables: int, initial_mode: int):
    _chk(_lib.moebius_bind(ctx, _vp(dev_base), _vp(dev_staging or None), _vp(dev_desc), _vp(dev_tables),
                           initial_mode), "moebius_bind")


def moebius_active_mode(ctx) -> int:
    return _lib.moebius_active_mode(ctx)


def _i32(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.int32)
    if shape is not None and a.shape != shape:
        raise ValueError("expected shape %r, got %r" % (shape, a.shape))
    return a


def moebius_plan(ctx, from_mode: int, to_mode: int, seq_lens, src_owner, src_block_tables):
    """seq_lens int32[n]; src_owner int32[n] or None; src_block_tables int32[n, max_pages]."""
    n = 0 if seq_lens is None else len(seq_lens)
    lens = _i32(seq_lens if n else np.zeros(0, np.int32))
    own = None if src_owner is None else _i32(src_owner, (n,))
    bt = _i32(src_block_tables if n else np.zeros((0, 1), np.int32))
    out = _vp()
    st = _lib.moebius_plan(ctx, from_mode, to_mode, n,
                           lens.ctypes.data_as(_vp) if n else None,
                           own.ctypes.data_as(_vp) if own is not None and n else None,
                           bt.ctypes.data_as(_vp) if n else None, C.byref(out))
    _chk(st, "moebius_plan")
    return out


def moebius_plan_destroy(plan):
    _lib.moebius_plan_destroy(plan)


def moebius_block_tables(plan, n_req: int, max_pages: int):
    owner = np.empty(n_req, np.int32)
    bt = np.empty((n_req, max_pages), np.int32)
    _chk(_lib.moebius_block_tables(plan, owner.ctypes.data_as(_vp), bt.ctypes.data_as(_vp)),
         "moebius_block_tables")
    return owner, bt


def moebius_plan_stats(plan) -> moebius_stats_t:
    out = moebius_stats_t()
    out.struct_size = C.sizeof(moebius_stats_t)
    _chk(_lib.moebius_plan_stats(plan, C.byref(out)), "moebius_plan_stats")
    return out


def moebius_plan_export(plan, what: int) -> np.ndarray:
    dt = (SEG_DTYPE, KV_DTYPE, C2D_DTYPE, np.dtype("<i4"), BULK_DTYPE, WBLK_DTYPE)[what]
    need = C.c_int64(0)
    _chk(_lib.moebius_plan_export(plan, what, None, 0, C.byref(need)), "moebius_plan_export")
    buf = np.zeros(need.value // dt.itemsize, dtype=dt)
    if need.value:
        _chk(_lib.moebius_plan_export(plan, what, buf.ctypes.data_as(_vp), need.value, C.byref(need)),
             "moebius_plan_export")
    return buf


def moebius_reshard(ctx, plan, cuda_stream: int = 0):
    _chk(_lib.moebius_reshard(ctx, plan, _vp(cuda_stream or None)), "moebius_reshard")


_lib.moebius_set_kv_slice.argtypes = [_vp, C.c_int]
_lib.moebius_set_chain_bands.argtypes = [_vp, C.c_int]
_lib.moebius_set_xt_mode.argtypes = [_vp, C.c_int]
_lib.moebius_reshard_shares.argtypes = [_vp, _vp, C.c_int, _vp, C.c_int, C.c_int, _vp]


def moebius_set_xt_mode(ctx, mode: int):
    _chk(_lib.moebius_set_xt_mode(ctx, mode), "moebius_set_xt_mode")


def moebius_set_chain_bands(ctx, enable: bool):
    _chk(_lib.moebius_set_chain_bands(ctx, 1 if enable else 0), "moebius_set_chain_bands")


def moebius_set_kv_slice(ctx, min_units: int):
    _chk(_lib.moebius_set_kv_slice(ctx, min_units), "moebius_set_kv_slice")


def moebius_reshard_shares(ctx, plan, rank_bounds, share_first: int, share_count: int, cuda_stream: int = 0):
    """One launch executing shares [share_first, share_first + share_count) of len(rank_bounds) - 1, all
    waves, with the device-side round barrier."""
    b = _i32(rank_bounds)
    _chk(_lib.moebius_reshard_shares(ctx, plan, len(b) - 1, b.ctypes.data_as(_vp), share_first, share_count,
                                     _vp(cuda_stream or None)), "moebius_reshard_shares")


_lib.moebius_naive_scratch_bytes.argtypes = [_vp, _vp, C.POINTER(C.c_int64)]
_lib.moebius_reshard_naive.argtypes = [_vp, _vp, _vp, C.c_int64, _vp, C.POINTER(C.c_int64)]


_lib.moebius_static_scratch_bytes.restype = C.c_int64
_lib.moebius_reshard_naive_static.argtypes = [_vp, _vp, _vp, C.POINTER(C.c_int64)]


def moebius_static_scratch_bytes() -> int:
    return int(_lib.moebius_static_scratch_bytes())


def moebius_reshard_naive_static(ctx, plan, cuda_stream: int = 0) -> dict:
    """moebius_reshard_naive with the library's static device scratch: allocates no device memory."""
    st = (C.c_int64 * 6)()
    _chk(_lib.moebius_reshard_naive_static(ctx, plan, _vp(cuda_stream or None), st), "moebius_reshard_naive_static")
    return {"launches": st[0], "bytes_read": st[1], "bytes_written": st[2], "w_pass_bytes": st[3],
            "kv_pass_bytes": st[4], "scratch_bytes": st[5]}


def moebius_naive_scratch_bytes(ctx, plan) -> int:
    out = C.c_int64(0)
    _chk(_lib.moebius_naive_scratch_bytes(ctx, plan, C.byref(out)), "moebius_naive_scratch_bytes")
    return out.value


def moebius_reshard_naive(ctx, plan, dev_scratch: int, scratch_bytes: int, cuda_stream: int = 0) -> dict:
    """The staged comparison path (Table 1); returns its launch / byte counts."""
    st = (C.c_int64 * 6)()
    _chk(_lib.moebius_reshard_naive(ctx, plan, _vp(dev_scratch), scratch_bytes, _vp(cuda_stream or None), st),
         "moebius_reshard_naive")
    return dict(zip(("launches", "bytes_read", "bytes_written", "w_pass_bytes", "kv_pass_bytes", "scratch_bytes"), list(st)))


def moebius_policy_preset(kind: int, T_h: float = 256.0, cooldown_s: float = 5.0) -> moebius_policy_config_t:
    out = moebius_policy_config_t()
    out.struct_size = C.sizeof(moebius_policy_config_t)
    _chk(_lib.moebius_policy_preset(kind, T_h, cooldown_s, C.byref(out)), "moebius_policy_preset")
    return out


def moebius_policy_config(T_h: float, T_l: float, W: int, cooldown_s: float) -> moebius_policy_config_t:
    out = moebius_policy_config_t()
    out.struct_size = C.sizeof(moebius_policy_config_t)
    out.T_h, out.T_l, out.W, out.cooldown_s = T_h, T_l, W, cooldown_s
    return out


def moebius_policy_create(cfg: moebius_policy_config_t, initial_mode: int):
    cfg.struct_size = C.sizeof(moebius_policy_config_t)
    out = _vp()
    _chk(_lib.moebius_policy_create(C.byref(cfg), initial_mode, C.byref(out)), "moebius_policy_create")
    return out


def moebius_policy_destroy(policy):
    _lib.moebius_policy_destroy(policy)


def moebius_policy_mode(policy) -> int:
    return _lib.moebius_policy_mode(policy)


def moebius_policy_step(policy, ctx, now_s: float, seq_lens):
    """Returns (decision, mode_after).  ctx may be None (no capacity check)."""
    lens = _i32(seq_lens if len(seq_lens) else np.zeros(0, np.int32))
    dec, mode = C.c_int32(0), C.c_int32(0)
    _chk(_lib.moebius_policy_step(policy, ctx, now_s, len(lens), lens.ctypes.data_as(_vp) if len(lens) else None,
                                  C.byref(dec), C.byref(mode)), "moebius_policy_step")
    return dec.value, mode.value


def moebius_capacity_check(ctx, to_mode: int, seq_lens) -> bool:
    lens = _i32(seq_lens if len(seq_lens) else np.zeros(0, np.int32))
    st = _lib.moebius_capacity_check(ctx, to_mode, len(lens), lens.ctypes.data_as(_vp) if len(lens) else None)
    if st == -2:
        return False
    _chk(st, "moebius_capacity_check")
    return True


def moebius_policy_calibrate(batch_sizes, tp_cost, ep_cost) -> int:
    b = _i32(batch_sizes)
    t = np.ascontiguousarray(tp_cost, np.float64)
    e = np.ascontiguousarray(ep_cost, np.float64)
    out = C.c_int32(0)
    _chk(_lib.moebius_policy_calibrate(len(b), b.ctypes.data_as(_vp), t.ctypes.data_as(_vp), e.ctypes.data_as(_vp),
                                       C.byref(out)), "moebius_policy_calibrate")
    return out.value


def moebius_plan_waves(plan) -> int:
    n = C.c_int32(0)
    _chk(_lib.moebius_plan_waves(plan, C.byref(n)), "moebius_plan_waves")
    return n.value


def moebius_share_stats(plan, rank_lo: int, rank_hi: int, wave: int = -1) -> dict:
    out = np.zeros(4, np.int64)
    _chk(_lib.moebius_share_stats(plan, rank_lo, rank_hi, wave, out.ctypes.data_as(_vp)), "moebius_share_stats")
    return {"units": int(out[0]), "read": int(out[1]), "written": int(out[2]), "cross": int(out[3])}


def moebius_reshard_share(ctx, plan, rank_lo: int, rank_hi: int, wave: int, cuda_stream: int = 0):
    _chk(_lib.moebius_reshard_share(ctx, plan, rank_lo, rank_hi, wave, _vp(cuda_stream or None)), "moebius_reshard_share")


def moebius_reshard_publish(ctx, plan, cuda_stream: int = 0):
    _chk(_lib.moebius_reshard_publish(ctx, plan, _vp(cuda_stream or None)), "moebius_reshard_publish")


def moebius_arena_create(ctx, device: int, rank_lo: int, rank_hi: int):
    out = _vp()
    _chk(_lib.moebius_arena_create(ctx, device, rank_lo, rank_hi, C.byref(out)), "moebius_arena_create")
    return out


def moebius_arena_destroy(arena):
    _lib.moebius_arena_destroy(arena)


def moebius_arena_base(arena) -> int:
    return int(_lib.moebius_arena_base(arena) or 0)


def moebius_arena_ready(arena) -> bool:
    return _lib.moebius_arena_ready(arena) == 0


def moebius_arena_export(arena, rank: int) -> int:
    fd = C.c_int32(-1)
    _chk(_lib.moebius_arena_export(arena, rank, C.byref(fd)), "moebius_arena_export")
    return fd.value


def moebius_arena_import(arena, rank: int, fd: int):
    _chk(_lib.moebius_arena_import(arena, rank, fd), "moebius_arena_import")


def moebius_stage_plan(ctx, plan):
    _chk(_lib.moebius_stage_plan(ctx, plan), "moebius_stage_plan")


def moebius_reshard_staged(ctx, cuda_stream: int = 0):
    _chk(_lib.moebius_reshard_staged(ctx, _vp(cuda_stream or None)), "moebius_reshard_staged")


def moebius_set_timing(ctx, enable: bool):
    _chk(_lib.moebius_set_timing(ctx, int(enable)), "moebius_set_timing")


def moebius_last_kernel_ms(ctx) -> float:
    ms = C.c_float(0)
    _chk(_lib.moebius_last_kernel_ms(ctx, C.byref(ms)), "moebius_last_kernel_ms")
    return ms.value


def moebius_kernel_ms_history(ctx, cap: int = 64):
    buf = (C.c_float * cap)()
    n = C.c_int(0)
    _chk(_lib.moebius_kernel_ms_history(ctx, buf, cap, C.byref(n)), "moebius_kernel_ms_history")
    return [buf[i] for i in range(n.value)]


def moebius_set_launch(ctx, ctas_per_sm: int = 0, threads: int = 0, unit_kb: int = 0):
    _chk(_lib.moebius_set_launch(ctx, ctas_per_sm, threads, unit_kb), "moebius_set_launch")


def moebius_set_tma(ctx, enable: bool = True, pipes: int = 0, stage_kb: int = 0):
    _chk(_lib.moebius_set_tma(ctx, int(enable), pipes, stage_kb), "moebius_set_tma")


def moebius_set_ring(ctx, ring_kb: int = 0, max_loads: int = 0):
    _chk(_lib.moebius_set_ring(ctx, ring_kb, max_loads), "moebius_set_ring")


def moebius_set_l2_policy(ctx, load_policy: int = 0, store_policy: int = 0):
    _chk(_lib.moebius_set_l2_policy(ctx, load_policy, store_policy), "moebius_set_l2_policy")


def moebius_set_kv_rounds(ctx, max_level: int = 0):
    _chk(_lib.moebius_set_kv_rounds(ctx, max_level), "moebius_set_kv_rounds")
