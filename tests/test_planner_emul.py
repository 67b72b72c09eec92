"""CPU tests of the product's host planner + unit decode through the test-only host emulator.
The emulator executes the exported work list with the product's own decode code on host memory and
checks every access against the ordering the device counters enforce; the result is compared with
the oracle bytewise.  (Device execution itself is covered by the -m gpu tests.)"""
import numpy as np
import pytest

import oracle
import workloads as wl
from harness import (EP, TP, OracleLayout, State, emulate, expected_attn_bytes, expected_bytes, expected_target, mb,
                     mb_config, source_tables)


def run_switch(st, sess, image, staging, from_mode, src_owner, src_bt):
    to_mode = EP if from_mode == TP else TP
    plan = sess.plan(to_mode, st.lens, src_owner, src_bt, from_mode=from_mode)
    stats = mb.moebius_plan_stats(plan).as_dict()
    owner, bt = sess.block_tables(plan, len(st.lens))
    want_owner, want_bt = expected_target(st, sess, to_mode)
    if to_mode == EP:
        assert np.array_equal(owner, want_owner)
    else:
        assert np.all(owner == -1)
    assert np.array_equal(bt, want_bt)
    res = emulate(sess, plan, image, staging)
    assert res["violations"] == 0 and res["oob"] == 0 and res["bad_wait"] == 0 and res["bad_begin"] == 0, res
    assert res["units"] == stats["n_units"]
    # byte accounting == oracle enumeration ("moves only the owner-changed bytes")
    ep_owner = src_owner if from_mode == EP else owner
    w, k = expected_bytes(st, from_mode, ep_owner)
    assert (stats["w_moved"], stats["w_relocated"], stats["w_read"]) == (w["moved"], w["relocated"], w["read"])
    assert (stats["kv_moved"], stats["kv_relocated"], stats["kv_read"]) == (k["moved"], k["relocated"], k["read"])
    assert (stats["attn_moved"], stats["attn_relocated"], stats["attn_read"]) == expected_attn_bytes(st, from_mode)
    direct_bytes = stats["w_relocated"] + stats["kv_relocated"] + stats["attn_relocated"]
    staged_extra = res["bytes_written"] - direct_bytes
    assert staged_extra >= 0
    if stats["n_kv_staged"] == 0:
        # EP->TP reads a straddled scale block once per holder: `read` counts unique source bytes (A15)
        rereads = stats["w_relocated"] - stats["w_read"]
        parked = stats["w_staged_bytes"]      # S2: a parked block is written to its slot and read back once more
        assert res["bytes_written"] == direct_bytes + parked
        assert res["bytes_read"] == stats["w_read"] + stats["kv_read"] + stats["attn_read"] + rereads + parked
    tgt = OracleLayout(st, sess, to_mode, want_owner, want_bt)
    bad = tgt.compare(image)
    assert not bad, bad[:5]
    sess.free_plan(plan)
    return to_mode, (want_owner if to_mode == EP else None), want_bt, stats


def make(cfg, lens=None, policy=None, cap_frac=0.0, pool_bytes=None):
    st = State(cfg, lens)
    sess = mb.Session(mb_config(cfg, st.lens, policy, cap_frac, pool_bytes))
    image = np.zeros(sess.layout.base_bytes, np.uint8)
    image[:] = 0xA5
    staging = np.full(max(sess.layout.staging_bytes, 16), 0x5A, np.uint8)
    return st, sess, image, staging


@pytest.mark.parametrize("src", ["canonical", "random"])
def test_tiny_round_trip(src):
    """TP -> EP -> TP on the tiny config: every view bit-exact after each switch, and the final TP
    bytes equal the initial ones on every valid byte."""
    st, sess, image, staging = make(wl.get_config("tiny"))
    owner, bt = source_tables(st, sess, TP, src)
    OracleLayout(st, sess, TP, owner, bt).place(image)
    mode, owner, bt, s1 = run_switch(st, sess, image, staging, TP, owner, bt)
    assert mode == EP
    mode, owner, bt, s2 = run_switch(st, sess, image, staging, EP, owner, bt)
    assert mode == TP
    assert s1["w_moved"] == s2["w_moved"] == 49152  # (1 - 1/2) * 3 * 8*64*32*2 bytes


SMALLISH = wl.get_config("small").with_(L=2, H=128, I=256, n_req=24, len_dist=("uniform", 1, 200), seed=77)


@pytest.mark.parametrize("first", [TP, EP])
@pytest.mark.parametrize("src", ["canonical", "random"])
def test_smallish_alternating(first, src):
    st, sess, image, staging = make(SMALLISH)
    mode = first
    owner, bt = source_tables(st, sess, mode, src)
    OracleLayout(st, sess, mode, owner, bt).place(image)
    for _ in range(3):
        mode, owner, bt, stats = run_switch(st, sess, image, staging, mode, owner, bt)


@pytest.mark.parametrize("R,Hkv", [(8, 4), (4, 4), (2, 8), (4, 1), (1, 2)])
def test_head_geometries(R, Hkv):
    """Replicated heads (Qwen3 4 heads on 8 ranks), Hkv == R (Fig. 8(b)), several
    heads per rank, a single head, and R = 1 (empty weight plan)."""
    cfg = wl.get_config("tiny").with_(R=R, E=8, I=64, kv_heads=Hkv, n_req=7, len_dist=("uniform", 1, 70), seed=5 + R)
    st, sess, image, staging = make(cfg)
    owner, bt = source_tables(st, sess, TP, "random")
    OracleLayout(st, sess, TP, owner, bt).place(image)
    mode, owner, bt, s1 = run_switch(st, sess, image, staging, TP, owner, bt)
    mode, owner, bt, s2 = run_switch(st, sess, image, staging, EP, owner, bt)
    if R == 1:
        assert s1["w_moved"] == 0 and s1["w_relocated"] == 0


def test_weight_only_warmup_switch():
    """n_req = 0: PAPER.md:199 'a weight-only warmup switch ... while no request is active'."""
    st, sess, image, staging = make(wl.get_config("tiny"), lens=[])
    OracleLayout(st, sess, TP, None, np.zeros((0, 1), np.int32)).place(image)
    mode, owner, bt, s = run_switch(st, sess, image, staging, TP, None, np.zeros((0, 1), np.int32))
    assert s["n_kv_moves"] == 0 and s["kv_moved"] == 0
    run_switch(st, sess, image, staging, EP, np.zeros(0, np.int32), np.zeros((0, 1), np.int32))


@pytest.mark.parametrize("first", [TP, EP])
def test_tight_pool_rounds_and_staging(first):
    """Tight pool: target pages overlap live source pages, so the plan needs dependency rounds and
    staging (BASELINE.json: 'in-place permutation cycles through a bounded staging buffer')."""
    cfg = SMALLISH.with_(L=1, n_req=40, seed=99)
    lens = wl.draw_seq_lens(cfg)
    seen_rounds = seen_staged = 0
    for seed in range(3):
        st, sess, image, staging = make(cfg, lens, "tight", cap_frac=0.5)
        mode = first
        owner, bt = source_tables(st, sess, mode, "random", seed=seed)
        OracleLayout(st, sess, mode, owner, bt).place(image)
        for _ in range(2):
            mode, owner, bt, stats = run_switch(st, sess, image, staging, mode, owner, bt)
            seen_rounds = max(seen_rounds, stats["n_kv_rounds"])
            seen_staged = max(seen_staged, stats["n_kv_staged"])
            assert stats["staging_used_bytes"] <= sess.layout.staging_bytes
    assert seen_rounds > 2 and seen_staged > 0


def test_staging_reused_across_pool_groups_and_too_small():
    """When the staged pages of all 2L pools do not fit the staging buffer, the pools are processed
    in groups that reuse it; when not even one pool fits, chains are cut less often; when the
    cycle-breaking pages alone do not fit, the plan fails with E_STAGING and the caller cancels
    the switch (like a capacity failure)."""
    cfg = SMALLISH.with_(L=2, n_req=40, seed=99)
    lens = wl.draw_seq_lens(cfg)
    st, sess, image, staging = make(cfg, lens, "tight", cap_frac=0.5)
    mb.moebius_set_kv_rounds(sess.ctx, 2)       # short schedules: chains are cut often, many staged pages
    owner, bt = source_tables(st, sess, TP, "random", seed=1)
    plan = sess.plan(EP, st.lens, owner, bt, from_mode=TP)
    s = mb.moebius_plan_stats(plan).as_dict()
    assert s["n_kv_staged"] > 0 and s["n_pool_groups"] == 1
    per_pool = s["n_kv_staged"] * sess.layout.ep_page_bytes
    spare = sess.layout.weight_spare_bytes
    # room for one pool's staged pages only -> 2L = 4 groups
    c = mb_config(cfg, lens, "tight")
    c.staging_cap_bytes = spare + per_pool + sess.layout.ep_page_bytes
    sess2 = mb.Session(c)
    mb.moebius_set_kv_rounds(sess2.ctx, 2)
    image = np.full(sess2.layout.base_bytes, 0xA5, np.uint8)
    staging = np.full(sess2.layout.staging_bytes, 0x5A, np.uint8)
    OracleLayout(st, sess2, TP, owner, bt).place(image)
    mode, o2, bt2, stats = run_switch(st, sess2, image, staging, TP, owner, bt)
    assert stats["n_pool_groups"] == 4 and stats["staging_used_bytes"] <= sess2.layout.staging_bytes
    run_switch(st, sess2, image, staging, EP, o2, bt2)
    # not even one pool's cut pages fit: the planner allows longer chains (fewer cuts, more rounds)
    c.staging_cap_bytes = spare + per_pool - sess.layout.ep_page_bytes
    sess3 = mb.Session(c)
    mb.moebius_set_kv_rounds(sess3.ctx, 2)
    image = np.full(sess3.layout.base_bytes, 0xA5, np.uint8)
    staging = np.full(sess3.layout.staging_bytes, 0x5A, np.uint8)
    OracleLayout(st, sess3, TP, owner, bt).place(image)
    _, _, _, stats3 = run_switch(st, sess3, image, staging, TP, owner, bt)
    assert stats3["n_kv_staged"] < s["n_kv_staged"] and stats3["n_kv_rounds"] >= s["n_kv_rounds"]
    assert stats3["staging_used_bytes"] <= sess3.layout.staging_bytes
    # no staging at all, but cycles need it: E_STAGING, the caller cancels the switch
    c.staging_cap_bytes = spare
    sess4 = mb.Session(c)
    assert sess4.layout.staging_bytes == 0
    with pytest.raises(mb.MoebiusError) as e:
        sess4.plan(EP, st.lens, owner, bt, from_mode=TP)
    assert e.value.status == -3
    # cap below the spare weight slot itself: no longer a refusal -- the views alias (shift 0) and the
    # weights take the in-place path, the cap going to staging
    c.staging_cap_bytes = spare - 1
    sess5 = mb.Session(c)
    assert sess5.layout.w_shift_slots == 0 and sess5.layout.weight_spare_bytes == 0
    assert 0 < sess5.layout.staging_bytes <= spare - 1
    st0 = State(cfg, [])                      # weight-only switches: all of it goes to the weights
    empty = np.zeros((0, 1), np.int32)
    image = np.full(sess5.layout.base_bytes, 0xA5, np.uint8)
    staging = np.full(sess5.layout.staging_bytes, 0x5A, np.uint8)
    OracleLayout(st0, sess5, TP, None, empty).place(image)
    _, o5, bt5, stats5 = run_switch(st0, sess5, image, staging, TP, None, empty)
    assert stats5["n_w_waves"] > 0 and stats5["n_w_parked"] > 0
    run_switch(st0, sess5, image, staging, EP, np.zeros(0, np.int32), empty)


def test_capacity_error_cancels_switch():
    """TP replication halves capacity; a switch that does not fit is cancelled."""
    cfg = wl.get_config("tiny").with_(R=4, I=64, kv_heads=2, n_req=6, len_dist=("uniform", 30, 64), seed=11)
    lens = wl.draw_seq_lens(cfg)
    pages = int(((lens + 15) // 16).sum())
    ep_page = 16 * 2 * 16 * 2
    # EP pools can hold every request of a rank, but the TP pool (same bytes, 2 heads on 4 ranks ->
    # each rank stores a replicated head) cannot hold all requests
    pool = ep_page * (pages // 2)
    st = State(cfg, lens)
    sess = mb.Session(mb_config(cfg, lens, pool_bytes=pool))
    assert sess.layout.pages_tp == 2 * sess.layout.pages_ep and sess.layout.pages_tp < pages
    owner, bt = source_tables(st, sess, EP, "canonical")
    with pytest.raises(mb.MoebiusError) as e:
        sess.plan(TP, st.lens, owner, bt, from_mode=EP)
    assert e.value.status == -2


def test_invalid_inputs():
    cfg = wl.get_config("tiny")
    lens = np.array([5, 20], np.int32)
    sess = mb.Session(mb_config(cfg, lens))
    bt = np.array([[0, -1], [1, 1]], np.int32)       # page 1 listed twice
    with pytest.raises(mb.MoebiusError) as e:
        sess.plan(EP, lens, None, bt, from_mode=TP)
    assert e.value.status == -1
    bt = np.array([[0, -1], [1, 9999]], np.int32)    # out of range
    with pytest.raises(mb.MoebiusError):
        sess.plan(EP, lens, None, bt, from_mode=TP)
    with pytest.raises(mb.MoebiusError):             # from == to
        sess.plan(TP, lens, None, bt, from_mode=TP)
    for bad in (dict(I=30), dict(E=7), dict(kv_heads=3, R=2)):
        with pytest.raises(mb.MoebiusError):
            mb.Session(mb_config(cfg.with_(**bad), lens))


def test_fp8_scales():
    cfg = wl.get_config("fp8_graph").with_(L=1, E=8, H=256, I=1536, n_req=6, len_dist=("uniform", 1, 60), seed=3)
    st, sess, image, staging = make(cfg)
    st.fill = "normal"
    owner, bt = source_tables(st, sess, TP, "random")
    OracleLayout(st, sess, TP, owner, bt).place(image)
    mode, owner, bt, s = run_switch(st, sess, image, staging, TP, owner, bt)
    mode, owner, bt, s = run_switch(st, sess, image, staging, EP, owner, bt)


@pytest.mark.parametrize("max_level", [1, 2, 6, 1024])
@pytest.mark.parametrize("first", [TP, EP])
def test_chain_cut_levels(first, max_level):
    """Dependency chains are cut by staging after `max_level` rounds (moebius_set_kv_rounds): the
    result and the hazard ordering are the same for every setting; only rounds vs staged pages trade."""
    cfg = SMALLISH.with_(L=1, n_req=40, seed=99)
    lens = wl.draw_seq_lens(cfg)
    st, sess, image, staging = make(cfg, lens, "tight", cap_frac=0.5)
    mb.moebius_set_kv_rounds(sess.ctx, max_level)
    owner, bt = source_tables(st, sess, first, "random", seed=2)
    OracleLayout(st, sess, first, owner, bt).place(image)
    mode, owner, bt, stats = run_switch(st, sess, image, staging, first, owner, bt)
    assert stats["n_kv_rounds"] <= max_level + 2
    if max_level == 1024:
        assert stats["n_kv_rounds"] > 8          # the uncut chains are long here
    run_switch(st, sess, image, staging, mode, owner, bt)
    sess.close()


# ---- the paper's own weight orientation (w_orient = 1) and odd shapes ----------------

@pytest.mark.parametrize("src", ["canonical", "random"])
def test_paper_orientation_tiny_round_trip(src):
    """W13 [E,2I,H] / W2 [E,H,I]: two chain objects of different size per layer (2 slots + 1 slot),
    EP views shifted by the larger one.  TP -> EP -> TP, every view bit-exact after each switch."""
    st, sess, image, staging = make(wl.get_config("tiny").with_(w_orient=1))
    assert sess.layout.weight_spare_bytes == 2 * sess.layout.weight_slot_bytes * st.cfg.R
    owner, bt = source_tables(st, sess, TP, src)
    OracleLayout(st, sess, TP, owner, bt).place(image)
    mode, owner, bt, s1 = run_switch(st, sess, image, staging, TP, owner, bt)
    mode, owner, bt, s2 = run_switch(st, sess, image, staging, EP, owner, bt)
    assert mode == TP and s1["w_moved"] == s2["w_moved"] == 49152


@pytest.mark.parametrize("first", [TP, EP])
def test_paper_orientation_smallish_alternating(first):
    st, sess, image, staging = make(SMALLISH.with_(w_orient=1))
    mode = first
    owner, bt = source_tables(st, sess, mode, "random")
    OracleLayout(st, sess, mode, owner, bt).place(image)
    for _ in range(3):
        mode, owner, bt, stats = run_switch(st, sess, image, staging, mode, owner, bt)


def test_paper_orientation_fp8_scales():
    cfg = wl.get_config("fp8_graph").with_(L=2, E=8, H=256, I=1536, n_req=6, len_dist=("uniform", 1, 60), seed=3,
                                           w_orient=1)
    st, sess, image, staging = make(cfg)
    st.fill = "normal"
    owner, bt = source_tables(st, sess, TP, "random")
    OracleLayout(st, sess, TP, owner, bt).place(image)
    mode, owner, bt, s = run_switch(st, sess, image, staging, TP, owner, bt)
    mode, owner, bt, s = run_switch(st, sess, image, staging, EP, owner, bt)


def test_paper_orientation_view_ids():
    """Tensor ids are per orientation: gate/up/down ids are invalid under w_orient = 1 and vice versa."""
    cfg = wl.get_config("tiny")
    lens = np.array([5], np.int32)
    s0 = mb.Session(mb_config(cfg, lens))
    s1 = mb.Session(mb_config(cfg.with_(w_orient=1), lens))
    for t in (mb.T_W13, mb.T_W2):
        with pytest.raises(mb.MoebiusError):
            s0.view_desc(TP, 0, 0, t)
    for t in (mb.T_GATE, mb.T_UP, mb.T_DOWN):
        with pytest.raises(mb.MoebiusError):
            s1.view_desc(TP, 0, 0, t)
    v = s1.view_desc(TP, 1, 0, mb.T_W13)
    assert tuple(v.shape[:3]) == (cfg.E, 2 * cfg.I // cfg.R, cfg.H)
    v = s1.view_desc(EP, 1, 0, mb.T_W2)
    assert tuple(v.shape[:3]) == (cfg.E // cfg.R, cfg.H, cfg.I)


@pytest.mark.parametrize("orient", [0, 1])
@pytest.mark.parametrize("R,E,H,I,Hkv", [(3, 6, 40, 72, 3), (6, 12, 24, 48, 2), (5, 10, 56, 40, 5)])
def test_non_power_of_two_shapes(orient, R, E, H, I, Hkv):
    """as an in-place transposition, non-power-of-two shapes give very long cycles; with
    shifted slots every object moves out of place, so nothing about the shape matters beyond reading
    A3 (E % R == 0, I % R == 0, 16-byte runs)."""
    cfg = wl.get_config("tiny").with_(R=R, L=2, E=E, H=H, I=I, kv_heads=Hkv, head_dim=24, n_req=9,
                                      len_dist=("uniform", 1, 90), seed=31 + R, w_orient=orient)
    st, sess, image, staging = make(cfg)
    owner, bt = source_tables(st, sess, TP, "random")
    OracleLayout(st, sess, TP, owner, bt).place(image)
    mode, owner, bt, _ = run_switch(st, sess, image, staging, TP, owner, bt)
    mode, owner, bt, _ = run_switch(st, sess, image, staging, EP, owner, bt)
    assert mode == TP


# ---- rank-share execution: the plan wave by wave (multi-GPU form) ----------

def wave_barrier_list(plan):
    """The exported work list re-ordered wave by wave, every wave waiting for ALL of the previous one
    (a barrier across GPUs): counter w is signalled by every segment of wave w."""
    segs = mb.moebius_plan_export(plan, 0).copy()
    waves = mb.moebius_plan_export(plan, 3)
    assert len(waves) == len(segs) and mb.moebius_plan_waves(plan) == (int(waves.max()) + 1 if len(waves) else 0)
    order = np.argsort(waves, kind="stable")
    out = segs[order]
    w_sorted = waves[order]
    units = np.array([int(out["n_units"][w_sorted == w].sum()) for w in range(int(w_sorted.max()) + 1)])
    out["signal_ctr"] = w_sorted
    out["wait_ctr"] = w_sorted - 1
    out["wait_target"] = np.where(w_sorted > 0, units[np.maximum(w_sorted - 1, 0)], 0)
    out["unit_begin"] = np.concatenate([[0], np.cumsum(out["n_units"])[:-1]])
    return out, w_sorted


@pytest.mark.parametrize("first", [TP, EP])
@pytest.mark.parametrize("policy,orient", [(None, 0), ("tight", 0), (None, 1)])
def test_waves_with_barriers_are_hazard_free(first, policy, orient):
    """Executing the plan wave by wave, with nothing ordered inside a wave, is hazard-free and gives the
    oracle's layout: this is what R GPUs do with one barrier per wave (moebius_reshard_share)."""
    import ctypes as C
    from harness import emul_lib
    cfg = SMALLISH.with_(L=2, n_req=30, seed=41, w_orient=orient)
    st, sess, image, staging = make(cfg, None, policy, cap_frac=0.5 if policy else 0.0)
    owner, bt = source_tables(st, sess, first, "random")
    OracleLayout(st, sess, first, owner, bt).place(image)
    to = EP if first == TP else TP
    plan = sess.plan(to, st.lens, owner, bt, from_mode=first)
    segs, w_sorted = wave_barrier_list(plan)
    # a dependent segment is always in a later wave than what it waits for
    orig = mb.moebius_plan_export(plan, 0)
    waves = mb.moebius_plan_export(plan, 3)
    for i, s in enumerate(orig):
        if s["wait_ctr"] >= 0:
            assert all(waves[j] < waves[i] for j in range(len(orig)) if orig[j]["signal_ctr"] == s["wait_ctr"])
    kv = mb.moebius_plan_export(plan, 1)
    c2d = mb.moebius_plan_export(plan, 2)
    bulk = mb.moebius_plan_export(plan, 4)
    wblk = mb.moebius_plan_export(plan, 5)
    out = np.zeros(8, np.int64)
    vp = lambda a: a.ctypes.data_as(C.c_void_p) if a.size else None  # noqa: E731
    emul_lib().emul_run(vp(image), image.size, vp(staging), staging.size, vp(segs), len(segs), vp(kv), vp(c2d),
                        sess.layout.rank_stride_bytes, vp(out), vp(bulk), vp(wblk), sess.w_staging_offset())
    assert out[0] == 0 and out[1] == 0 and out[2] == 0 and out[3] == 0, out
    want_owner, want_bt = expected_target(st, sess, to)
    assert not OracleLayout(st, sess, to, want_owner, want_bt).compare(image)
    sess.free_plan(plan)


@pytest.mark.parametrize("first", [TP, EP])
@pytest.mark.parametrize("R,Hkv", [(8, 4), (4, 8), (4, 4)])
def test_share_stats_partition_the_plan(first, R, Hkv):
    """The rank shares are a disjoint cover of the plan, wave by wave, and the bytes that cross between
    ranks sum to the owner-changed bytes (oracle/accounting.py enumerates them)."""
    cfg = SMALLISH.with_(R=R, E=16, kv_heads=Hkv, L=2, n_req=20, seed=51)
    st, sess, image, staging = make(cfg)
    owner, bt = source_tables(st, sess, first, "random")
    to = EP if first == TP else TP
    plan = sess.plan(to, st.lens, owner, bt, from_mode=first)
    stats = mb.moebius_plan_stats(plan).as_dict()
    new_owner, _ = sess.block_tables(plan, len(st.lens))
    w, k = expected_bytes(st, first, owner if first == EP else new_owner)
    per_rank = [mb.moebius_share_stats(plan, r, r + 1) for r in range(R)]
    assert sum(s["units"] for s in per_rank) == stats["n_units"]
    assert sum(s["cross"] for s in per_rank) == w["moved"] + k["moved"] == stats["w_moved"] + stats["kv_moved"]
    if stats["n_kv_staged"] == 0:
        assert sum(s["written"] for s in per_rank) == w["relocated"] + k["relocated"]
        assert sum(s["read"] for s in per_rank) == w["read"] + k["read"]
    whole = mb.moebius_share_stats(plan, 0, R)
    assert whole == {key: sum(s[key] for s in per_rank) for key in whole}
    n_waves = mb.moebius_plan_waves(plan)
    by_wave = [mb.moebius_share_stats(plan, 0, R, wv) for wv in range(n_waves)]
    assert sum(s["units"] for s in by_wave) == stats["n_units"] and all(s["units"] > 0 for s in by_wave)
    # weights are balanced across ranks by construction; every rank has work in every weight wave
    assert all(mb.moebius_share_stats(plan, r, r + 1, 0)["units"] > 0 for r in range(R))
    sess.free_plan(plan)


@pytest.mark.parametrize("attn_mode", [1, 2])
@pytest.mark.parametrize("R,Hq,Hkv", [(2, 4, 2), (4, 8, 2), (4, 8, 8), (8, 16, 4), (1, 4, 2), (3, 6, 3)])
def test_attention_projections_follow_the_switch(attn_mode, R, Hq, Hkv):
    """default variant (both layouts resident: the switch moves nothing, both sets of
    views hold the oracle's layouts at all times) and the memory-saving variant (TP shard in place
    inside the full tensor; TP->EP gathers the other ranks' shards, EP->TP keeps the local slice)."""
    cfg = wl.get_config("tiny").with_(R=R, E=R * 2, I=16 * R, kv_heads=Hkv, n_q_heads=Hq, attn_mode=attn_mode, L=2,
                                       n_req=5, len_dist=("uniform", 1, 40), seed=40 + R)
    st, sess, image, staging = make(cfg)
    lay = sess.layout
    a = oracle.attn_bytes(R, cfg.L, Hq, Hkv, cfg.head_dim, cfg.H, 2, "tp2ep", "dual" if attn_mode == 1 else "gather")
    assert lay.attn_full_bytes == a["full_per_rank"] * R
    assert lay.attn_dup_bytes == a["duplicated_per_rank"] * R
    owner, bt = source_tables(st, sess, TP, "random")
    src = OracleLayout(st, sess, TP, owner, bt)
    src.place(image)
    mode = TP
    for _ in range(3):
        mode, owner, bt, stats = run_switch(st, sess, image, staging, mode, owner, bt)
        if attn_mode == 1:   # pointer swap: compare() has checked BOTH modes' views; nothing moved
            assert stats["attn_moved"] == 0
    sess.close()


S2_CASES = {
    # name: (config, staging cap as a fraction of resident bytes or 0)
    "tiny_inplace": (wl.get_config("tiny").with_(w_inplace=1), 0.0),
    "small_inplace": (SMALLISH.with_(w_inplace=1, seed=81), 0.0),
    "odd_shape_inplace": (wl.get_config("tiny").with_(R=3, E=6, H=40, I=72, kv_heads=3, head_dim=8, n_req=9,
                                                       len_dist=("uniform", 1, 90), seed=21, w_inplace=1), 0.0),
    "E60_R4_inplace": (wl.get_config("tiny").with_(R=4, E=60, H=24, I=32, kv_heads=4, n_req=5, seed=22, w_inplace=1), 0.0),
    "paper_orient_inplace": (SMALLISH.with_(w_orient=1, w_inplace=1, seed=82), 0.0),
    "paper_orient_shift1": (SMALLISH.with_(w_orient=1, seed=83, L=3), -1.95),     # cap = 1.95 objects: one spare slot, not two
    "fp8_inplace": (wl.get_config("fp8_graph").with_(L=2, E=8, H=256, I=1536, n_req=6, len_dist=("uniform", 1, 60), seed=3,
                                                     w_inplace=1), 0.0),
    "R5_inplace": (wl.get_config("tiny").with_(R=5, E=10, H=16, I=40, kv_heads=5, n_req=4, seed=23, w_inplace=1), 0.0),
}


@pytest.mark.parametrize("name", sorted(S2_CASES))
@pytest.mark.parametrize("first", [TP, EP])
def test_s2_in_place_path(name, first):
    """SURVEY.md section 7 S2 / BASELINE.json north_star: when the cap leaves no room for a spare slot as
    large as the largest object, the EP and TP views overlap (down to aliasing the same bytes) and the
    move becomes an in-place permutation: blocks in dependency waves, blocks on cycles parked in the
    bounded staging buffer.  Hazard-free under the emulator and bit-exact with the oracle, both ways."""
    cfg, cap = S2_CASES[name]
    st = State(cfg, fill="normal" if cfg.w_dtype == "fp8_e4m3_b128" else "tag")
    if cap < 0:        # given in units of one object over all ranks
        probe = mb.Session(mb_config(cfg, st.lens))
        cap = -cap * probe.layout.weight_slot_bytes * cfg.R / probe.layout.resident_bytes
        probe.close()
    sess = mb.Session(mb_config(cfg, st.lens, None, cap))
    lay = sess.layout
    max_obj = 2 if cfg.w_orient else 1
    assert lay.w_shift_slots < max_obj and lay.w_staging_bytes > 0
    assert lay.weight_spare_bytes == lay.w_shift_slots * lay.weight_slot_bytes * cfg.R
    if cap:
        assert lay.weight_spare_bytes + lay.staging_bytes <= cap * lay.resident_bytes
    image = np.full(lay.base_bytes, 0xA5, np.uint8)
    staging = np.full(max(lay.staging_bytes, 16), 0x5A, np.uint8)
    owner, bt = source_tables(st, sess, first, "random")
    OracleLayout(st, sess, first, owner, bt).place(image)
    mode = first
    waves = parked = 0
    for _ in range(3):
        mode, owner, bt, stats = run_switch(st, sess, image, staging, mode, owner, bt)
        waves, parked = max(waves, stats["n_w_waves"]), max(parked, stats["n_w_parked"])
        assert stats["w_staged_bytes"] <= stats["w_relocated"]
    assert waves > 0
    if lay.w_shift_slots == 0:
        assert parked > 0          # aliased views: nothing can start before something is parked
    sess.close()


def necklaces(k, n):
    """Number of necklaces of length n over k symbols = size of a minimum feedback vertex set of the de
    Bruijn graph B(k, n) (Mykkeltveit 1972): (1/n) * sum over d | n of phi(d) * k^(n/d)."""
    phi = lambda d: sum(1 for a in range(1, d + 1) if np.gcd(a, d) == 1)   # noqa: E731
    return sum(phi(d) * k ** (n // d) for d in range(1, n + 1) if n % d == 0) // n


@pytest.mark.parametrize("name,R,words", [("qwen3_235b", 8, 3), ("qwen3_30b", 8, 3), ("small", 4, 4)])
def test_aliased_views_park_a_minimum_feedback_vertex_set(name, R, words):
    """Aliased views of a power-of-two shape cut into 64 blocks per rank: block (q, i) is blocked by the blocks
    at position (q*64 + i) div R of every rank -- the de Bruijn graph on R-ary words (q, digits of i).  What
    the planner parks per gate/up object is a feedback vertex set of it, and its greedy finds the minimum,
    the necklace count (176 of 512 at R = 8; 70 of 256 at R = 4), where taking the blockers of whichever block
    needs the fewest parks parked 260-324.  Host only: the plan's statistics."""
    cfg = wl.get_config(name).with_(w_inplace=1, n_req=0)
    assert cfg.R == R and R ** words == R * 64
    lens = np.zeros(0, np.int32)
    c = mb_config(cfg, wl.draw_seq_lens(wl.get_config(name)))
    c.max_requests = 1
    probe = mb.Session(c)
    c.staging_cap_bytes = int(0.024 * probe.layout.resident_bytes)
    probe.close()
    sess = mb.Session(c)
    per_down = None
    for to, frm in ((EP, TP), (TP, EP)):
        plan = sess.plan(to, lens, None if to == EP else np.zeros(0, np.int32), np.zeros((0, 1), np.int32), from_mode=frm)
        st = mb.moebius_plan_stats(plan).as_dict()
        sess.free_plan(plan)
        short = 2 * cfg.L * necklaces(R, words)              # gate and up of every layer
        down = st["n_w_parked"] - short                       # the long-run objects have fewer, larger blocks
        assert down > 0 and down % cfg.L == 0 and down // cfg.L < necklaces(R, words), (st["n_w_parked"], short)
        per_down = per_down or down
        assert down == per_down                               # the same both ways
        # parked bytes (every parked block moves twice): 34-41 % of the weights, not 53-63 %
        assert st["w_staged_bytes"] < 0.45 * st["w_relocated"]
    sess.close()


def test_s2_is_chosen_by_the_cap_and_refuses_only_what_cannot_fit():
    """The planner picks the shift from staging_cap_bytes: S1 (every move out of place) when a spare of
    the largest object fits, else fewer slots plus the in-place path; E_STAGING only when not even the
    duplicated attention shards fit."""
    cfg = SMALLISH.with_(w_orient=1, L=3, seed=83)
    lens = wl.draw_seq_lens(cfg)
    probe = mb.Session(mb_config(cfg, lens))
    res, S = probe.layout.resident_bytes, probe.layout.weight_slot_bytes * cfg.R
    assert probe.layout.w_shift_slots == 2          # no cap: S1
    probe.close()
    seen = set()
    for cap in (2.2 * S, 2 * S, 1.99 * S, 1.3 * S, S, 0.5 * S, 1):
        c = mb_config(cfg, lens)
        c.staging_cap_bytes = int(cap)
        s = mb.Session(c)
        lay = s.layout
        seen.add(lay.w_shift_slots)
        assert lay.weight_spare_bytes + lay.staging_bytes <= max(int(cap), lay.weight_spare_bytes)
        assert lay.w_staging_bytes == 0 if lay.w_shift_slots == 2 else (lay.w_staging_bytes > 0 or cap < S)
        if cap == 1:     # a cap that leaves no staging at all: the in-place path cannot park anything -> cancelled
            bt = wl.random_page_tables(lens, None, cfg.R, lay.pages_tp, cfg.page, c.max_pages_per_request, seed=1)
            with pytest.raises(mb.MoebiusError) as e:
                s.plan(EP, lens, None, bt, from_mode=TP)
            assert e.value.status == -3
        s.close()
    assert seen == {0, 1, 2}
    assert res > 0


@pytest.mark.parametrize("first", [TP, EP])
def test_banded_chain_overlaps_links_and_the_checker_sees_a_wrong_band(first):
    """Equal-sized objects, every move out of place: each chain link is cut into 2 x 2 segments that wait
    for ONE half of the predecessor (moebius_set_chain_bands).  The emulator finds the schedule hazard-free
    -- and finds violations when the two halves a link waits for are swapped (negative control: the
    checker does see a wrong band), or when the waits are dropped."""
    import ctypes as C
    from harness import emul_lib
    cfg = SMALLISH.with_(L=3, seed=55)
    st, sess, image, staging = make(cfg)
    mb.moebius_set_chain_bands(sess.ctx, True)
    owner, bt = source_tables(st, sess, first, "random")
    src = OracleLayout(st, sess, first, owner, bt)
    src.place(image)
    to = EP if first == TP else TP
    plan = sess.plan(to, st.lens, owner, bt, from_mode=first)
    segs = mb.moebius_plan_export(plan, 0)
    w = segs[(segs["kind"] & 0xFF) == 0]
    n_links = cfg.L * 3
    assert len(w) == 4 * n_links and np.all(w["n_desc"] == cfg.R // 2)          # (regular) block lists of R/2 blocks
    assert np.all(w["stg_pools"] == 1) and len(mb.moebius_plan_export(plan, 5)) == 0   # no descriptors
    assert len(set(w["signal_ctr"].tolist())) == 2 * n_links                     # two counters per link
    first_link, later = w[:4], w[4:]
    assert np.all(first_link["wait_ctr"] == -1) and np.all(later["wait_ctr"] >= 0)
    # every later segment waits for exactly one of its predecessor's two counters
    for i in range(1, n_links):
        prev_ctrs = set(w[4 * (i - 1):4 * i]["signal_ctr"].tolist())
        assert set(w[4 * i:4 * i + 4]["wait_ctr"].tolist()) == prev_ctrs
    # unbanded for comparison: one segment per link
    sess_u = mb.Session(sess.cfg)          # the default: unbanded
    plan_u = sess_u.plan(to, st.lens, owner, bt, from_mode=first)
    wu = mb.moebius_plan_export(plan_u, 0)
    assert int(((wu["kind"] & 0xFF) == 0).sum()) == n_links
    sess_u.close()

    def run(tampered):
        img = image.copy()
        stg = staging.copy()
        out = np.zeros(8, np.int64)
        vp = lambda a: a.ctypes.data_as(C.c_void_p) if a.size else None  # noqa: E731
        kv, c2d, bulk, wblk = (mb.moebius_plan_export(plan, k) for k in (1, 2, 4, 5))
        emul_lib().emul_run(vp(img), img.size, vp(stg), stg.size, vp(tampered), len(tampered), vp(kv), vp(c2d),
                            sess.layout.rank_stride_bytes, vp(out), vp(bulk), vp(wblk), sess.w_staging_offset())
        return out

    assert run(segs)[0] == 0 and run(segs)[2] == 0
    swapped = segs.copy()
    idx = np.flatnonzero((segs["kind"] & 0xFF) == 0)
    for i in range(1, n_links):                      # make each segment wait for the OTHER half
        blk = idx[4 * i:4 * i + 4]
        a, b = sorted(set(segs["wait_ctr"][blk].tolist()))
        units = {int(c): int(t) for c, t in zip(segs["wait_ctr"][blk], segs["wait_target"][blk])}
        for j in blk:
            other = b if segs["wait_ctr"][j] == a else a
            swapped["wait_ctr"][j] = other
            swapped["wait_target"][j] = units[other]
    assert run(swapped)[0] > 0
    dropped = segs.copy()
    dropped["wait_ctr"][idx] = -1
    assert run(dropped)[0] > 0
    sess.free_plan(plan)
    sess.close()
