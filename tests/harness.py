"""Shared test harness: builds the logical state (workloads), its oracle layouts (oracle), places
the SOURCE layout at the library's view offsets in a byte image, and compares the TARGET layout the
product produced (GPU, or the host emulator in CPU tests) with the oracle, bytewise on every view
and in the block tables.  The oracle never sees product output; the product never sees the oracle."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

import oracle
import paper_2606_26607_b200 as mb
import workloads as wl

HERE = os.path.dirname(os.path.abspath(__file__))
KINDS = ("gate", "up", "down")
TP, EP = mb.MOEBIUS_TP, mb.MOEBIUS_EP
MODE = {TP: "tp", EP: "ep"}


def mb_config(cfg: wl.Config, seq_lens, pool_policy=None, staging_cap_frac=0.0, pool_bytes=None,
              max_requests=None, max_pages=None):
    pool = pool_bytes if pool_bytes is not None else wl.kv_pool_bytes(cfg, seq_lens, pool_policy)
    n = len(seq_lens)
    mp = max_pages or max(1, int(max([0] + [(int(x) + cfg.page - 1) // cfg.page for x in seq_lens])))
    c = mb.make_config(R=cfg.R, L=cfg.L, E=cfg.E, H=cfg.H, I=cfg.I, w_dtype=cfg.w_dtype,
                       kv_heads=cfg.kv_heads, head_dim=cfg.head_dim, page_tokens=cfg.page,
                       kv_pool_bytes_per_rank_layer=pool, max_requests=max_requests or max(n, 1),
                       max_pages_per_request=mp, staging_cap_bytes=0, w_orient=cfg.w_orient,
                       n_q_heads=cfg.n_q_heads, attn_mode=cfg.attn_mode, w_inplace=cfg.w_inplace)
    if staging_cap_frac:
        s = mb.Session(c)
        c.staging_cap_bytes = int(staging_cap_frac * s.layout.resident_bytes)
        s.close()
    return c


State = oracle.State


def view_fn_of(sess: mb.Session):
    def fn(mode, rank, layer, tensor_id):
        v = sess.view_desc(mode, rank, layer, tensor_id)
        return (v.offset, tuple(v.shape[i] for i in range(v.ndim)), v.elem_bytes,
                tuple(v.stride[i] for i in range(v.ndim)))
    return fn


def OracleLayout(st, sess: mb.Session, mode: int, owner, bt):
    return oracle.OracleLayout(st, view_fn_of(sess), sess.layout.pages_tp, sess.layout.pages_ep, mode, owner, bt)


def source_tables(st: State, sess: mb.Session, mode: int, how: str, seed: int = 7):
    """(owner, bt) of the SOURCE mode.  how = 'canonical' (oracle reading A7) or 'random' (A8)."""
    c = st.cfg
    lay = sess.layout
    mp = sess.cfg.max_pages_per_request
    owner = oracle.partition_requests(st.lens, c.R) if mode == EP else None
    n_pages = lay.pages_ep if mode == EP else lay.pages_tp
    if how == "canonical":
        bt = oracle.canonical_block_tables(st.lens, owner, MODE[mode], n_pages, c.page, mp)
    else:
        bt = wl.random_page_tables(st.lens, owner, c.R, n_pages, c.page, mp, seed)
    return owner, bt


def expected_target(st: State, sess: mb.Session, to_mode: int):
    """Oracle request state after the switch: owner and canonical tables (A7)."""
    return oracle.target_request_state(st, to_mode, sess.layout.pages_tp, sess.layout.pages_ep,
                                       sess.cfg.max_pages_per_request)


def expected_bytes(st: State, from_mode: int, ep_owner):
    c = st.cfg
    d = "ep2tp" if from_mode == EP else "tp2ep"
    w = oracle.weight_bytes(c.R, c.L, c.E, c.H, c.I, c.w_elem_bytes, d) if c.R > 1 else \
        {"moved": 0, "relocated": 0, "read": 0}
    if c.w_dtype == "fp8_e4m3_b128":      # the block scales travel with their weights (reading A13)
        s = oracle.scale_bytes(c.R, c.L, c.E, c.H, c.I, d, c.w_kinds)
        w = {key: w[key] + s[key] for key in w}
    k = oracle.kv_bytes(st.lens, ep_owner if ep_owner is not None else np.zeros(len(st.lens), np.int32),
                        c.R, c.L, c.kv_heads, c.head_dim, c.kv_elem_bytes, d)
    return w, k


def expected_attn_bytes(st: State, from_mode: int):
    """(moved, relocated, read) of the attention projections (oracle/attention.py)."""
    c = st.cfg
    if not c.attn_mode:
        return (0, 0, 0)
    a = oracle.attn_bytes(c.R, c.L, c.n_q_heads, c.kv_heads, c.head_dim, c.H, 2,
                          "ep2tp" if from_mode == EP else "tp2ep", "dual" if c.attn_mode == 1 else "gather")
    return (a["moved"], a["relocated"], a["read"])


# ---- host emulator (CPU tests only) ---------------------------------------------------------------

_EMUL = None


def emul_lib():
    global _EMUL
    if _EMUL is None:
        src = os.path.join(HERE, "emul", "emul.cpp")
        so = os.path.join(HERE, "emul", "libemul.so")
        hdr = os.path.join(HERE, "..", "paper_2606_26607_b200", "csrc", "moebius_units.h")
        if (not os.path.exists(so)) or os.path.getmtime(so) < max(os.path.getmtime(src), os.path.getmtime(hdr)):
            subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", so, src])
        _EMUL = C.CDLL(so)
        _EMUL.emul_run.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_int64, C.c_void_p, C.c_int,
                                   C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64]
    return _EMUL


def emulate(sess: mb.Session, plan, image: np.ndarray, staging: np.ndarray):
    """Runs the exported work list through the product's unit decode on host memory, checking
    every access against the wait/signal ordering.  Returns the checker's counters."""
    segs = mb.moebius_plan_export(plan, 0)
    kv = mb.moebius_plan_export(plan, 1)
    c2d = mb.moebius_plan_export(plan, 2)
    bulk = mb.moebius_plan_export(plan, 4)
    wblk = mb.moebius_plan_export(plan, 5)
    out = np.zeros(8, np.int64)
    vp = lambda a: a.ctypes.data_as(C.c_void_p) if a.size else None  # noqa: E731
    emul_lib().emul_run(vp(image), image.size, vp(staging), staging.size, vp(segs), len(segs), vp(kv), vp(c2d),
                        sess.layout.rank_stride_bytes, vp(out), vp(bulk), vp(wblk), sess.w_staging_offset())
    return {"violations": int(out[0]), "oob": int(out[1]), "bad_wait": int(out[2]), "bad_begin": int(out[3]),
            "bytes_read": int(out[4]), "bytes_written": int(out[5]), "units": int(out[6])}
