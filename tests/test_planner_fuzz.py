"""Seeded fuzz of the host planner + unit decode through the hazard-checking emulator: random rank
counts, shapes (power of two or not), head geometries, dtypes, orientations, pool tightness, request
sets and source tables.  Every plan must be hazard-free, stay in bounds, move exactly the
owner-changed bytes the oracle enumerates, and leave the oracle's target layout -- in both
directions.  No GPU."""
import numpy as np
import pytest

import workloads as wl
from harness import (EP, TP, OracleLayout, State, emulate, expected_attn_bytes, expected_bytes, expected_target, mb, mb_config,
                     source_tables)


def draw_case(seed):
    rng = np.random.default_rng(1000 + seed)
    R = int(rng.choice([1, 2, 3, 4, 6, 8]))
    heads = [h for h in (1, 2, 3, 4, 6, 8, 12) if h % R == 0 or R % h == 0]
    Hkv = int(rng.choice(heads))
    w_dtype = str(rng.choice(["bf16", "bf16", "fp32", "fp8_e4m3_b128"]))
    eb = {"bf16": 2, "fp32": 4, "fp8_e4m3_b128": 1}[w_dtype]
    if w_dtype == "fp8_e4m3_b128":
        H = 128 * int(rng.integers(1, 3))
        I = 128 * R * int(rng.integers(1, 3)) if rng.random() < 0.5 else 192 * R     # 192: shards straddle blocks
        if I % 128:
            I = 128 * R
    else:
        H = 8 * int(rng.integers(1, 12))
        I = R * (16 // eb) * int(rng.integers(1, 7))
    cfg = wl.get_config("tiny").with_(
        R=R, L=int(rng.integers(1, 4)), E=R * int(rng.integers(1, 4)), H=H, I=I, w_dtype=w_dtype,
        kv_heads=Hkv, head_dim=8 * int(rng.integers(1, 5)), page=int(rng.choice([4, 16])),
        n_req=int(rng.integers(0, 14)), len_dist=("uniform", 1, int(rng.integers(2, 120))), seed=500 + seed,
        w_orient=int(rng.integers(0, 2)))
    # attention projections: none / both layouts resident / memory-saving All-Gather
    mult = [m for m in (1, 2, 4, 8) if (Hkv * m) % R == 0]
    attn_mode = int(rng.choice([0, 1, 2])) if mult else 0
    if attn_mode:
        cfg = cfg.with_(attn_mode=attn_mode, n_q_heads=Hkv * int(rng.choice(mult)))
    if rng.random() < 0.25:      # aliased EP / TP views: the in-place weight path (S2)
        cfg = cfg.with_(w_inplace=1)
    policy = str(rng.choice(["roomy", "tight"]))
    first = int(rng.choice([TP, EP]))
    src = str(rng.choice(["canonical", "random"]))
    rounds = int(rng.choice([0, 1, 3]))
    return cfg, policy, first, src, rounds


@pytest.mark.parametrize("seed", range(160))
def test_fuzz_round_trip(seed):
    cfg, policy, first, src, rounds = draw_case(seed)
    st = State(cfg, fill="normal" if cfg.w_dtype == "fp8_e4m3_b128" else "tag")
    try:
        sess = mb.Session(mb_config(cfg, st.lens, policy, 0.5 if policy == "tight" else 0.0))
    except mb.MoebiusError as e:       # a cap below the spare slot of this shape: a legal refusal
        assert e.status == -3
        return
    if rounds:
        mb.moebius_set_kv_rounds(sess.ctx, rounds)
    if seed % 3 == 0:
        mb.moebius_set_chain_bands(sess.ctx, True)      # the banded weight chain (off by default)
    image = np.full(sess.layout.base_bytes, 0xA5, np.uint8)
    staging = np.full(max(sess.layout.staging_bytes, 16), 0x5A, np.uint8)
    mode = first
    owner, bt = source_tables(st, sess, mode, src, seed=seed)
    OracleLayout(st, sess, mode, owner, bt).place(image)
    for _ in range(2):
        to = EP if mode == TP else TP
        try:
            plan = sess.plan(to, st.lens, owner, bt, from_mode=mode)
        except mb.MoebiusError as e:   # staging too small for the cycles of this draw: cancelled, nothing touched
            assert e.status == -3 and (policy == "tight" or cfg.w_inplace)
            return
        stats = mb.moebius_plan_stats(plan).as_dict()
        res = emulate(sess, plan, image, staging)
        assert (res["violations"], res["oob"], res["bad_wait"], res["bad_begin"]) == (0, 0, 0, 0), (seed, res)
        assert res["units"] == stats["n_units"]
        new_owner, new_bt = sess.block_tables(plan, len(st.lens))
        want_owner, want_bt = expected_target(st, sess, to)
        assert np.array_equal(new_bt, want_bt)
        assert np.array_equal(new_owner, want_owner if to == EP else np.full(len(st.lens), -1, np.int32))
        w, k = expected_bytes(st, mode, owner if mode == EP else new_owner)
        assert (stats["w_moved"], stats["w_relocated"], stats["w_read"]) == (w["moved"], w["relocated"], w["read"])
        assert (stats["kv_moved"], stats["kv_relocated"], stats["kv_read"]) == (k["moved"], k["relocated"], k["read"])
        assert (stats["attn_moved"], stats["attn_relocated"], stats["attn_read"]) == expected_attn_bytes(st, mode)
        shares = [mb.moebius_share_stats(plan, r, r + 1) for r in range(cfg.R)]
        assert sum(s["units"] for s in shares) == stats["n_units"]
        assert sum(s["cross"] for s in shares) == stats["w_moved"] + stats["kv_moved"] + stats["attn_moved"]
        bad = OracleLayout(st, sess, to, want_owner, want_bt).compare(image)
        assert not bad, (seed, bad[:3])
        sess.free_plan(plan)
        owner, bt, mode = (want_owner if to == EP else None), want_bt, to
    sess.close()
