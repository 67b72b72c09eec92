"""GPU parity: the sm_100a reshard kernel, called through the C ABI, against the CPU oracle.

Every case places the oracle's SOURCE layout at the library's fixed view offsets, uploads it, runs
`moebius_plan` + `moebius_reshard` on the device, downloads the unified buffer and compares the
TARGET layout bytewise with what the oracle builds from the logical tensors (bit-exact: it is byte
movement), plus the block tables and the owner vector.  Guard strips round
every caller-owned buffer must come back untouched.
"""
import numpy as np
import pytest

import workloads as wl
from harness import (EP, TP, OracleLayout, State, expected_attn_bytes, expected_bytes, expected_target, mb, mb_config,
                     source_tables)

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

GUARD = 4096
CANARY = 0xC3


def gpu_session(cfg, lens=None, policy=None, cap_frac=0.0, pool_bytes=None, fill="tag", initial_mode=TP, tma=None,
                vmm=False):
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (there is no CPU fallback)"
    st = State(cfg, lens, fill=fill)
    sess = mb.Session(mb_config(cfg, st.lens, policy, cap_frac, pool_bytes), device="cuda:0", guard_bytes=GUARD,
                      initial_mode=initial_mode, vmm=vmm)
    if tma is not None:
        mb.moebius_set_tma(sess.ctx, *tma)
    sess.arena.fill_(CANARY)
    return st, sess


def upload(sess, image):
    sess.base[:image.size].copy_(torch.from_numpy(image))


def download(sess):
    torch.cuda.synchronize()
    return sess.base.cpu().numpy()


def check_guards(sess):
    for i, g in enumerate(sess.guards()):
        assert bool((g == CANARY).all()), "guard strip %d was written" % i


def device_tables(sess, n_req):
    """What the captured graphs read: header, owner, lens and block tables at their fixed address."""
    lay = sess.layout
    t = sess.tables.cpu().numpy()
    mr, mp = sess.cfg.max_requests, sess.cfg.max_pages_per_request
    hdr = t[:16]
    owner = t[lay.tbl_owner_off:lay.tbl_owner_off + mr]
    lens = t[lay.tbl_lens_off:lay.tbl_lens_off + mr]
    bt = t[lay.tbl_bt_off:lay.tbl_bt_off + n_req * mp].reshape(n_req, mp)
    return hdr, owner, lens, bt


def gpu_switch(st, sess, from_mode, src_owner, src_bt, execute=None):
    to_mode = EP if from_mode == TP else TP
    plan = sess.plan(to_mode, st.lens, src_owner, src_bt, from_mode=from_mode)
    stats = mb.moebius_plan_stats(plan).as_dict()
    owner, bt = sess.block_tables(plan, len(st.lens))
    want_owner, want_bt = expected_target(st, sess, to_mode)
    if execute is None:
        sess.reshard(plan)
    else:
        execute(sess, plan)
    got = download(sess)
    assert mb.moebius_active_mode(sess.ctx) == to_mode
    # tables: host copy and the published device copy, bit-exact with the oracle
    if to_mode == EP:
        assert np.array_equal(owner, want_owner)
    else:
        assert np.all(owner == -1)
    assert np.array_equal(bt, want_bt)
    n = len(st.lens)
    hdr, d_owner, d_lens, d_bt = device_tables(sess, n)
    assert hdr[0] == to_mode and hdr[1] == n
    assert np.array_equal(d_bt, want_bt)
    assert np.array_equal(d_lens[:n], st.lens)
    assert np.array_equal(d_owner[:n], want_owner if to_mode == EP else np.full(n, -1, np.int32))
    # every view of the target mode, bytewise
    bad = OracleLayout(st, sess, to_mode, want_owner, want_bt).compare(got)
    assert not bad, bad[:5]
    check_guards(sess)
    # accounting
    ep_owner = src_owner if from_mode == EP else owner
    w, k = expected_bytes(st, from_mode, ep_owner)
    assert (stats["w_moved"], stats["w_relocated"], stats["w_read"]) == (w["moved"], w["relocated"], w["read"])
    assert (stats["kv_moved"], stats["kv_relocated"], stats["kv_read"]) == (k["moved"], k["relocated"], k["read"])
    assert (stats["attn_moved"], stats["attn_relocated"], stats["attn_read"]) == expected_attn_bytes(st, from_mode)
    sess.free_plan(plan)
    return to_mode, (want_owner if to_mode == EP else None), want_bt, stats


def start(st, sess, mode, how, seed=7):
    owner, bt = source_tables(st, sess, mode, how, seed=seed)
    image = np.full(sess.layout.base_bytes, 0xA5, np.uint8)
    OracleLayout(st, sess, mode, owner, bt).place(image)
    upload(sess, image)
    return owner, bt, image


@pytest.mark.parametrize("src", ["canonical", "random"])
def test_tiny_round_trip(src):
    """BASELINE.json config 1: TP -> EP -> TP; the final TP views equal the initial ones."""
    st, sess = gpu_session(wl.get_config("tiny"))
    owner, bt, image0 = start(st, sess, TP, src)
    mode, owner, bt, _ = gpu_switch(st, sess, TP, owner, bt)
    mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt)
    assert mode == TP
    # the weights' TP views sit at the same fixed addresses as before: bytes identical
    got = download(sess)
    c = st.cfg
    for r in range(c.R):
        for m in range(3):
            v = sess.view_desc(TP, r, 0, m)
            n = int(np.prod([v.shape[i] for i in range(v.ndim)])) * v.elem_bytes
            assert np.array_equal(got[v.offset:v.offset + n], image0[v.offset:v.offset + n])
    sess.close()


SMALLISH = wl.get_config("small").with_(L=2, H=128, I=256, n_req=24, len_dist=("uniform", 1, 200), seed=77)


@pytest.mark.parametrize("first", [TP, EP])
def test_smallish_alternating(first):
    st, sess = gpu_session(SMALLISH, initial_mode=first)
    mode = first
    owner, bt, _ = start(st, sess, mode, "random")
    for _ in range(4):
        mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt)
    sess.close()


@pytest.mark.parametrize("R,Hkv", [(8, 4), (4, 4), (2, 8), (4, 1), (1, 2)])
def test_head_geometries(R, Hkv):
    cfg = wl.get_config("tiny").with_(R=R, E=8, I=64, kv_heads=Hkv, n_req=7, len_dist=("uniform", 1, 70), seed=5 + R)
    st, sess = gpu_session(cfg)
    owner, bt, _ = start(st, sess, TP, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, TP, owner, bt)
    mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt)
    sess.close()


def test_weight_only_warmup_switch():
    """n_req = 0."""
    st, sess = gpu_session(wl.get_config("tiny"), lens=[])
    empty = np.zeros((0, 1), np.int32)
    image = np.full(sess.layout.base_bytes, 0xA5, np.uint8)
    OracleLayout(st, sess, TP, None, empty).place(image)
    upload(sess, image)
    mode, owner, bt, s = gpu_switch(st, sess, TP, None, empty)
    assert s["n_kv_moves"] == 0
    gpu_switch(st, sess, mode, np.zeros(0, np.int32), empty)
    sess.close()


@pytest.mark.parametrize("first", [TP, EP])
def test_tight_pool_rounds_and_staging(first):
    """Target pages overlap live source pages: dependency rounds + bounded staging on the device."""
    cfg = SMALLISH.with_(L=1, n_req=40, seed=99)
    lens = wl.draw_seq_lens(cfg)
    rounds = staged = 0
    for seed in range(3):
        st, sess = gpu_session(cfg, lens, "tight", cap_frac=0.5, initial_mode=first)
        mode = first
        owner, bt, _ = start(st, sess, mode, "random", seed=seed)
        for _ in range(2):
            mode, owner, bt, stats = gpu_switch(st, sess, mode, owner, bt)
            rounds, staged = max(rounds, stats["n_kv_rounds"]), max(staged, stats["n_kv_staged"])
        sess.close()
    assert rounds > 2 and staged > 0


def test_fp8_scales():
    cfg = wl.get_config("fp8_graph").with_(L=1, E=8, H=256, I=1536, n_req=6, len_dist=("uniform", 1, 60), seed=3)
    st, sess = gpu_session(cfg, fill="normal")
    owner, bt, _ = start(st, sess, TP, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, TP, owner, bt)
    mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt)
    sess.close()


def test_small_config_alternating():
    """BASELINE.json config 2 (R=4, 4 layers, E=16, H=1024, I=512; 64 requests of 128-2048 tokens):
    alternating TP->EP and EP->TP switches; spans many tiles of every segment kind and ragged tails."""
    cfg = wl.get_config("small")
    st, sess = gpu_session(cfg)
    mode = TP
    owner, bt, _ = start(st, sess, mode, "random")
    for _ in range(2):
        mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt)
    sess.close()


@pytest.mark.parametrize("threads,ctas,unit_kb", [(128, 1, 4), (256, 2, 64), (64, 8, 16)])
def test_launch_shapes(threads, ctas, unit_kb):
    """ld/st path only (TMA off): the result does not depend on the launch shape or the unit size."""
    st, sess = gpu_session(SMALLISH, initial_mode=EP, tma=(0, 0, 0))
    mb.moebius_set_launch(sess.ctx, ctas, threads, unit_kb)
    owner, bt, _ = start(st, sess, EP, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, EP, owner, bt)
    gpu_switch(st, sess, mode, owner, bt)
    sess.close()


@pytest.mark.parametrize("pipes,stage_kb", [(1, 96), (2, 48), (4, 24), (8, 8), (2, 16)])
@pytest.mark.parametrize("first", [TP, EP])
def test_tma_shapes(first, pipes, stage_kb):
    """TMA path: the result does not depend on the number of pipes or the stage size (which sets the
    rows per tensor-map box and the pools per KV unit); ragged last row blocks and partial pages."""
    st, sess = gpu_session(SMALLISH, initial_mode=first, tma=(1, pipes, stage_kb))
    owner, bt, _ = start(st, sess, first, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, first, owner, bt)
    gpu_switch(st, sess, mode, owner, bt)
    sess.close()


@pytest.mark.parametrize("pipes,stage_kb,ring_kb,max_loads", [
    (2, 48, 96, 1), (2, 48, 96, 2), (2, 48, 48, 1), (4, 24, 52, 3), (2, 16, 100, 6), (3, 32, 68, 7), (1, 24, 200, 7),
    (8, 8, 26, 2), (2, 40, 41, 1)])
@pytest.mark.parametrize("which", ["smallish", "small_tight", "inplace"])
def test_ring_shapes(which, pipes, stage_kb, ring_kb, max_loads):
    """The pipes' rings (moebius_set_ring): a unit takes the bytes it needs, first in first out, so rings
    that are no multiple of a unit (wrap padding), rings of exactly one unit, mixed unit sizes (weight
    boxes, bulk chunks, 1-3 KV pages, staged pages, parked blocks) and up to 7 loads in flight per pipe
    must all give the same bytes."""
    cfg = {"smallish": SMALLISH, "small_tight": wl.get_config("small").with_(L=2, n_req=24),
           "inplace": wl.get_config("small").with_(w_inplace=1, L=2, n_req=16)}[which]
    kw = dict(policy="tight", cap_frac=0.5) if which == "small_tight" else {}
    st, sess = gpu_session(cfg, initial_mode=TP, tma=(1, pipes, stage_kb), **kw)
    mb.moebius_set_ring(sess.ctx, ring_kb, max_loads)
    owner, bt, _ = start(st, sess, TP, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, TP, owner, bt)
    mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt)
    gpu_switch(st, sess, mode, owner, bt)
    sess.close()


@pytest.mark.parametrize("load_policy,store_policy", [(0, 0), (1, 1), (2, 0), (3, 4), (4, 2)])
def test_l2_policies(load_policy, store_policy):
    """moebius_set_l2_policy: cache hints on every TMA operation change no byte."""
    st, sess = gpu_session(wl.get_config("small").with_(L=1, n_req=12))
    mb.moebius_set_l2_policy(sess.ctx, load_policy, store_policy)
    owner, bt, _ = start(st, sess, TP, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, TP, owner, bt)
    gpu_switch(st, sess, mode, owner, bt)
    with pytest.raises(mb.MoebiusError):
        mb.moebius_set_l2_policy(sess.ctx, 5, 0)
    sess.close()


def test_ring_arguments():
    st, sess = gpu_session(SMALLISH, tma=(1, 2, 48))
    for bad in ((47, 1), (105, 1), (96, 8), (-1, 0)):      # below a stage, over 208 KB in all, too deep
        with pytest.raises(mb.MoebiusError):
            mb.moebius_set_ring(sess.ctx, *bad)
    mb.moebius_set_ring(sess.ctx, 0, 0)
    sess.close()


@pytest.mark.parametrize("pipes,stage_kb", [(2, 48), (4, 24), (2, 16)])
@pytest.mark.parametrize("first", [TP, EP])
@pytest.mark.parametrize("which", ["smallish", "small", "ragged", "inplace"])
def test_tp_side_box(which, first, pipes, stage_kb):
    """moebius_set_xt_mode(ctx, 1): the EP side of a short-run weight unit is one contiguous bulk copy and
    the tensor-map box covers the TP views.  Identical results; ragged last row blocks (rows per rank not a
    multiple of the box) fall back to the EP-side box unit by unit; block lists (banded chain, in-place
    path) use it too."""
    cfg = {"smallish": SMALLISH, "small": wl.get_config("small").with_(L=2, n_req=20),
           "ragged": wl.get_config("tiny").with_(R=4, E=12, H=50, I=128, kv_heads=4, n_req=6, seed=31),
           "inplace": wl.get_config("small").with_(w_inplace=1, L=2, n_req=16)}[which]
    st, sess = gpu_session(cfg, initial_mode=first, tma=(1, pipes, stage_kb))
    mb.moebius_set_xt_mode(sess.ctx, 1)
    owner, bt, _ = start(st, sess, first, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, first, owner, bt)
    mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt)
    mb.moebius_set_xt_mode(sess.ctx, 0)
    gpu_switch(st, sess, mode, owner, bt)
    sess.close()


@pytest.mark.parametrize("tma", [0, 1])
def test_small_config_both_paths(tma):
    """BASELINE.json config 2 on the ld/st path and on the TMA path: identical results."""
    cfg = wl.get_config("small")
    st, sess = gpu_session(cfg, tma=(tma, 0, 0))
    owner, bt, _ = start(st, sess, TP, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, TP, owner, bt)
    gpu_switch(st, sess, mode, owner, bt)
    sess.close()


def test_state_errors():
    st, sess = gpu_session(wl.get_config("tiny"))
    owner, bt, _ = start(st, sess, TP, "canonical")
    plan = sess.plan(TP, st.lens, *source_tables(st, sess, EP, "canonical"), from_mode=EP)
    with pytest.raises(mb.MoebiusError) as e:     # active mode is TP, plan.from is EP
        sess.reshard(plan)
    assert e.value.status == -4
    sess.close()


# ---- the paper's own weight orientation (w_orient = 1) and odd shapes ----------------

@pytest.mark.parametrize("tma", [0, 1])
def test_paper_orientation_small_config(tma):
    """Config 2 shapes with W13 [E,2I,H] / W2 [E,H,I]: chain objects of 2 slots + 1 slot per layer."""
    cfg = wl.get_config("small").with_(w_orient=1)
    st, sess = gpu_session(cfg, tma=(tma, 0, 0))
    owner, bt, _ = start(st, sess, TP, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, TP, owner, bt)
    gpu_switch(st, sess, mode, owner, bt)
    sess.close()


@pytest.mark.parametrize("first", [TP, EP])
def test_paper_orientation_tiny_and_fp8(first):
    st, sess = gpu_session(wl.get_config("tiny").with_(w_orient=1), initial_mode=first)
    owner, bt, _ = start(st, sess, first, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, first, owner, bt)
    gpu_switch(st, sess, mode, owner, bt)
    sess.close()
    cfg = wl.get_config("fp8_graph").with_(L=2, E=8, H=256, I=1536, n_req=6, len_dist=("uniform", 1, 60), seed=3,
                                           w_orient=1)
    st, sess = gpu_session(cfg, fill="normal", initial_mode=first)
    owner, bt, _ = start(st, sess, first, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, first, owner, bt)
    gpu_switch(st, sess, mode, owner, bt)
    sess.close()


@pytest.mark.parametrize("orient", [0, 1])
@pytest.mark.parametrize("R,E,H,I,Hkv", [(3, 6, 40, 72, 3), (6, 12, 24, 48, 2), (5, 10, 56, 40, 5)])
def test_non_power_of_two_shapes(orient, R, E, H, I, Hkv):
    """Shifted slots move every object out of place: odd rank counts and shapes need nothing special
    (as an in-place transposition they would give very long cycles)."""
    cfg = wl.get_config("tiny").with_(R=R, L=2, E=E, H=H, I=I, kv_heads=Hkv, head_dim=24, n_req=9,
                                      len_dist=("uniform", 1, 90), seed=31 + R, w_orient=orient)
    st, sess = gpu_session(cfg)
    owner, bt, _ = start(st, sess, TP, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, TP, owner, bt)
    mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt)
    assert mode == TP
    sess.close()


# ---- peer-mappable unified buffer: one virtual range, one physical allocation per rank (NEXT-1) ----

@pytest.mark.parametrize("name,orient", [("tiny", 0), ("small", 0), ("small", 1)])
def test_vmm_arena_round_trip(name, orient):
    """Every rank region is its own physical allocation mapped at base + r * rank_stride (PAPER.md:158,
    :172: exported once, mapped by peers); planner, kernel and tensor maps run unchanged on it."""
    cfg = wl.get_config(name).with_(w_orient=orient)
    st, sess = gpu_session(cfg, vmm=True)
    assert sess.layout.rank_stride_bytes % (2 << 20) == 0
    owner, bt, _ = start(st, sess, TP, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, TP, owner, bt)
    mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt)
    assert mode == TP
    sess.close()


def test_vmm_arena_export_import():
    """Arena B creates ranks [0, R/2) itself and imports ranks [R/2, R) from arena A through POSIX file
    descriptors (what a process does with its peers' regions).  A switch executed on B's range must be
    visible through A's mapping of the shared ranks: same physical bytes, two virtual addresses."""
    cfg = wl.get_config("small").with_(L=2, H=128, I=256, n_req=24, len_dist=("uniform", 1, 200), seed=77)
    st, sess = gpu_session(cfg)            # plain session: used for its context and side buffers
    R, half = cfg.R, cfg.R // 2
    stride = sess.layout.rank_stride_bytes
    A = mb.moebius_arena_create(sess.ctx, 0, half, R)
    B = mb.moebius_arena_create(sess.ctx, 0, 0, half)
    assert not mb.moebius_arena_ready(A) and not mb.moebius_arena_ready(B)
    import os
    for r in range(half, R):
        fd = mb.moebius_arena_export(A, r)
        mb.moebius_arena_import(B, r, fd)
        os.close(fd)
    assert mb.moebius_arena_ready(B)
    with pytest.raises(mb.MoebiusError):
        mb.moebius_arena_export(B, R - 1)   # not B's own allocation
    from paper_2606_26607_b200.session import _RawCuda
    baseB = torch.as_tensor(_RawCuda(mb.moebius_arena_base(B), int(sess.layout.base_bytes)), device="cuda:0")
    upperA = torch.as_tensor(_RawCuda(mb.moebius_arena_base(A) + half * stride, int((R - half) * stride)), device="cuda:0")
    mb.moebius_bind(sess.ctx, baseB.data_ptr(), sess.staging.data_ptr(), sess.desc.data_ptr(), sess.tables.data_ptr(), TP)
    sess.base = baseB
    owner, bt, _ = start(st, sess, TP, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, TP, owner, bt)
    torch.cuda.synchronize()
    assert torch.equal(upperA, baseB[half * stride:])
    assert int((upperA != 0xA5).sum()) > 0
    del baseB, upperA
    sess.base = None
    sess.close()
    mb.moebius_arena_destroy(B)
    mb.moebius_arena_destroy(A)


def share_execute(ranks_per_share):
    """The multi-GPU form on one GPU: wave by wave, the shares of a wave enqueued one after another (on
    R GPUs they run concurrently, with a barrier across GPUs after each wave), then publish."""
    def run(sess, plan):
        R = sess.cfg.R
        stream = torch.cuda.current_stream().cuda_stream
        for wave in range(mb.moebius_plan_waves(plan)):
            for lo in range(0, R, ranks_per_share):
                mb.moebius_reshard_share(sess.ctx, plan, lo, min(R, lo + ranks_per_share), wave, stream)
        mb.moebius_reshard_publish(sess.ctx, plan, stream)
    return run


@pytest.mark.parametrize("ranks_per_share", [1, 2])
@pytest.mark.parametrize("first", [TP, EP])
def test_rank_share_execution(first, ranks_per_share):
    """NEXT-1: every GPU executes only the units of the ranks it owns, one launch per dependency wave.
    Bit-identical to the fused launch: both must equal the oracle.  Runs on a VMM arena (one physical
    allocation per rank), from random tables in a tight pool (rounds + staging) and back."""
    cfg = wl.get_config("small").with_(L=2, H=128, I=256, n_req=30, len_dist=("uniform", 1, 200), seed=61)
    st, sess = gpu_session(cfg, None, "tight", cap_frac=0.5, initial_mode=first, vmm=True)
    owner, bt, _ = start(st, sess, first, "random")
    mode, owner, bt, s1 = gpu_switch(st, sess, first, owner, bt, execute=share_execute(ranks_per_share))
    mode, owner, bt, s2 = gpu_switch(st, sess, mode, owner, bt, execute=share_execute(ranks_per_share))
    assert mode == first and max(s1["n_kv_rounds"], s2["n_kv_rounds"]) > 1
    sess.close()


def test_rank_share_execution_fp8_replicated_heads():
    cfg = wl.get_config("fp8_graph").with_(L=2, E=8, H=256, I=1536, n_req=12, len_dist=("uniform", 1, 90), seed=3)
    st, sess = gpu_session(cfg, fill="normal", vmm=True)
    owner, bt, _ = start(st, sess, TP, "random")
    mode, owner, bt, _ = gpu_switch(st, sess, TP, owner, bt, execute=share_execute(1))
    mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt, execute=share_execute(4))
    sess.close()


# ---- seeded fuzz on the device: the same draws as tests/test_planner_fuzz.py -------------------------

@pytest.mark.parametrize("seed", range(0, 160, 5))
def test_fuzz_round_trip_on_device(seed):
    from test_planner_fuzz import draw_case
    cfg, policy, first, src, rounds = draw_case(seed)
    st = State(cfg, fill="normal" if cfg.w_dtype == "fp8_e4m3_b128" else "tag")
    try:
        c = mb_config(cfg, st.lens, policy, 0.5 if policy == "tight" else 0.0)
        sess = mb.Session(c, device="cuda:0", guard_bytes=GUARD, initial_mode=first, vmm=bool(seed % 2))
    except mb.MoebiusError as e:
        assert e.status == -3
        return
    if rounds:
        mb.moebius_set_kv_rounds(sess.ctx, rounds)
    sess.arena.fill_(CANARY)
    owner, bt, _ = start(st, sess, first, src, seed=seed)
    mode = first
    for k in range(2):
        try:
            mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt,
                                            execute=share_execute(1) if seed % 3 == 0 else None)
        except mb.MoebiusError as e:
            assert e.status == -3 and policy == "tight"
            break
    sess.close()


def test_first_switch_after_bind_allocates_nothing():
    """"a switch does not allocate dynamic buffers".  Everything one-off (timing events,
    the driver entry point, the tensor maps, the kernel's shared-memory attribute, module loading) is
    done by moebius_bind; the very FIRST moebius_reshard of a context -- and every later one -- leaves
    the free device memory and the host heap (glibc mallinfo2: arena + mmapped bytes in use) exactly as
    they were.  The plan (host object, pinned upload image) is built before the measured call."""
    import ctypes as C

    class Mallinfo2(C.Structure):
        _fields_ = [(n, C.c_size_t) for n in ("arena", "ordblks", "smblks", "hblks", "hblkhd", "usmblks", "fsmblks",
                                                "uordblks", "fordblks", "keepcost")]
    libc = C.CDLL("libc.so.6")
    libc.mallinfo2.restype = Mallinfo2

    def heap():
        m = libc.mallinfo2()
        return m.uordblks + m.hblkhd

    cfg = SMALLISH.with_(L=1)
    st, sess = gpu_session(cfg)
    mb.moebius_set_timing(sess.ctx, True)
    owner, bt, _ = start(st, sess, TP, "random")
    stream = torch.cuda.current_stream().cuda_stream
    mode = TP
    for k in range(3):
        to = EP if mode == TP else TP
        plan = sess.plan(to, st.lens, owner, bt, from_mode=mode)
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        h0 = heap()
        mb.moebius_reshard(sess.ctx, plan, stream)          # the measured call: ctypes straight into the C ABI
        h1 = heap()
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        assert free1 == free0, ("device memory changed during switch %d" % k, free0 - free1)
        assert h1 == h0, ("host heap changed during switch %d" % k, h1 - h0)
        want_owner, want_bt = expected_target(st, sess, to)
        assert not OracleLayout(st, sess, to, want_owner, want_bt).compare(download(sess))
        sess.free_plan(plan)
        owner, bt, mode = (want_owner if to == EP else None), want_bt, to
    assert mb.moebius_last_kernel_ms(sess.ctx) > 0
    sess.close()


def test_reshard_checks_come_before_the_first_enqueue():
    """include/moebius.h: a failed call leaves the context and all device bytes untouched.  A plan built
    for another stage geometry (moebius_set_tma after moebius_plan) is refused with E_STATE before
    anything is enqueued: the descriptor buffer, the tables and the data keep their bytes."""
    st, sess = gpu_session(SMALLISH.with_(L=1))
    owner, bt, _ = start(st, sess, TP, "random")
    plan = sess.plan(EP, st.lens, owner, bt, from_mode=TP)
    mb.moebius_set_tma(sess.ctx, 1, 1, 64)      # the default stage here is one 32-KB EP page
    torch.cuda.synchronize()
    before = sess.arena.clone()
    with pytest.raises(mb.MoebiusError) as e:
        sess.reshard(plan)
    assert e.value.status == -4
    torch.cuda.synchronize()
    assert torch.equal(before, sess.arena)
    assert mb.moebius_active_mode(sess.ctx) == TP
    # a plan built for the new geometry runs
    sess.free_plan(plan)
    gpu_switch(st, sess, TP, owner, bt)
    sess.close()


@pytest.mark.parametrize("attn_mode", [mb.ATTN_DUAL, mb.ATTN_GATHER])
@pytest.mark.parametrize("R,Hq,Hkv,D,H", [(8, 16, 4, 64, 256), (4, 8, 8, 32, 128), (2, 4, 1, 16, 64), (3, 6, 3, 8, 40)])
def test_attention_projections(attn_mode, R, Hq, Hkv, D, H):
    """SURVEY.md section 8(f) NEXT-4.  MOEBIUS_ATTN_DUAL: both layouts resident, a switch
    moves nothing and both sets of views stay bit-exact with the oracle.  MOEBIUS_ATTN_GATHER: the head
    shard sits in place inside the full tensor (wo as a strided view); TP->EP gathers the other ranks'
    shards on the device (bulk 2-D copies in the fused launch), EP->TP keeps the local slice."""
    cfg = wl.get_config("tiny").with_(R=R, E=2 * R, H=H, I=32 * R, kv_heads=Hkv, head_dim=D, n_q_heads=Hq,
                                       attn_mode=attn_mode, L=3, n_req=9, len_dist=("uniform", 1, 80), seed=60 + R)
    st, sess = gpu_session(cfg)
    owner, bt, _ = start(st, sess, TP, "random")
    mode = TP
    for _ in range(3):
        mode, owner, bt, stats = gpu_switch(st, sess, mode, owner, bt)
    if attn_mode == mb.ATTN_GATHER:
        # the strided TP view of wo, read through torch, equals the oracle's dense head shard
        sess2_mode = mode
        for r in range(R):
            got = sess.view(TP, r, 1, mb.T_WO).cpu().numpy().view(np.uint16)
            want = oracle_attn_tp(st, 1, "wo", r)
            if sess2_mode == TP:
                assert np.array_equal(got, want)
    sess.close()


def oracle_attn_tp(st, layer, kind, r):
    import oracle
    c = st.cfg
    return oracle.attn_tp_view(st.attn(layer, kind), kind, r, c.R, c.n_q_heads, c.kv_heads)


def naive_execute(sess, plan):
    """The staged comparison path (Table 1) instead of the fused kernel, same plan."""
    n = mb.moebius_naive_scratch_bytes(sess.ctx, plan)
    scratch = torch.empty(n + 512, dtype=torch.uint8, device="cuda:0")
    off = (-scratch.data_ptr()) % 256
    scratch[:off].fill_(CANARY)
    scratch[off + n:].fill_(CANARY)
    st = mb.moebius_reshard_naive(sess.ctx, plan, scratch.data_ptr() + off, n, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert bool((scratch[:off] == CANARY).all()) and bool((scratch[off + n:] == CANARY).all()), "naive path wrote outside its scratch"
    ps = mb.moebius_plan_stats(plan).as_dict()
    # Table 1 on one device: every weight byte makes 2 read+write passes, every KV byte 3
    assert st["w_pass_bytes"] == 2 * (ps["w_relocated"] - scale_relocated(sess, plan))
    assert st["kv_pass_bytes"] == 2 * ps["kv_read"] + (ps["kv_read"] + ps["kv_relocated"]) + 2 * ps["kv_relocated"]
    return st


def scale_relocated(sess, plan):
    c2d = mb.moebius_plan_export(plan, 2)
    return int((c2d["rows"].astype(np.int64) * c2d["run_bytes"]).sum())


NAIVE_CASES = {
    "tiny": wl.get_config("tiny"),
    "smallish": SMALLISH,
    "replicated_heads": wl.get_config("tiny").with_(R=8, E=8, I=64, kv_heads=4, n_req=7, len_dist=("uniform", 1, 70), seed=13),
    "one_head": wl.get_config("tiny").with_(R=4, E=8, I=64, kv_heads=1, n_req=7, len_dist=("uniform", 1, 70), seed=9),
    "fp8": wl.get_config("fp8_graph").with_(L=1, E=8, H=256, I=1536, n_req=6, len_dist=("uniform", 1, 60), seed=3),
    "paper_orient": SMALLISH.with_(w_orient=1, seed=78),
    "odd": wl.get_config("tiny").with_(R=3, E=6, H=40, I=72, kv_heads=3, head_dim=8, n_req=9, len_dist=("uniform", 1, 90), seed=21),
    "attn_gather": wl.get_config("tiny").with_(R=4, E=8, H=128, I=128, kv_heads=2, head_dim=32, n_q_heads=8, attn_mode=2, L=2,
                                               n_req=9, len_dist=("uniform", 1, 80), seed=64),
}


@pytest.mark.parametrize("name", sorted(NAIVE_CASES))
@pytest.mark.parametrize("first", [TP, EP])
def test_naive_three_stage_path_is_bit_exact(name, first):
    """SURVEY.md section 8(f) NEXT-4 (ii), Table 1: permute -> exchange (-> scatter)
    through a staging buffer gives the same target layout, tables and accounting as the fused kernel --
    compared with the same oracle -- and a fused switch can follow a staged one on the same buffer."""
    cfg = NAIVE_CASES[name]
    st, sess = gpu_session(cfg, fill="normal" if cfg.w_dtype == "fp8_e4m3_b128" else "tag", initial_mode=first)
    owner, bt, _ = start(st, sess, first, "random")
    mode = first
    for k in range(4):
        mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt, execute=naive_execute if k != 2 else None)
    sess.close()


def test_naive_path_with_tight_pools_needs_no_rounds():
    """Gathering a pool's live pages into the staging buffer first reads every source page before any
    target page is written: the staged path is hazard-free for any tables, at the price of its passes."""
    cfg = SMALLISH.with_(L=1, n_req=40, seed=99)
    st, sess = gpu_session(cfg, wl.draw_seq_lens(cfg), "tight", cap_frac=0.5)
    owner, bt, _ = start(st, sess, TP, "random", seed=1)
    mode = TP
    for _ in range(3):
        mode, owner, bt, stats = gpu_switch(st, sess, mode, owner, bt, execute=naive_execute)
    sess.close()


S2_GPU_CASES = {
    "tiny_inplace": (wl.get_config("tiny").with_(w_inplace=1), 0.0),
    "smallish_inplace": (SMALLISH.with_(w_inplace=1, seed=81), 0.0),
    "small_config_inplace": (wl.get_config("small").with_(w_inplace=1, L=2, n_req=16), 0.0),     # XT boxes inside blocks
    "odd_shape_inplace": (wl.get_config("tiny").with_(R=3, E=6, H=40, I=72, kv_heads=3, head_dim=8, n_req=9,
                                                       len_dist=("uniform", 1, 90), seed=21, w_inplace=1), 0.0),
    "E60_R4_inplace": (wl.get_config("tiny").with_(R=4, E=60, H=24, I=32, kv_heads=4, n_req=5, seed=22, w_inplace=1), 0.0),
    "paper_orient_shift1": (SMALLISH.with_(w_orient=1, seed=83, L=3), -1.95),
    "paper_orient_inplace": (SMALLISH.with_(w_orient=1, w_inplace=1, seed=82), 0.0),
    "fp8_inplace": (wl.get_config("fp8_graph").with_(L=2, E=8, H=256, I=1536, n_req=6, len_dist=("uniform", 1, 60), seed=3,
                                                     w_inplace=1), 0.0),
}


@pytest.mark.parametrize("name", sorted(S2_GPU_CASES))
@pytest.mark.parametrize("first", [TP, EP])
def test_s2_in_place_path_on_device(name, first):
    """SURVEY.md section 7 S2 on the device: aliased (or partly overlapping) EP / TP views, blocks in
    dependency waves, blocks on permutation cycles parked in the bounded staging buffer -- including a
    non-power-of-two shape (E = 60, R = 4; R = 3) -- bit-exact with the oracle in both directions."""
    cfg, cap = S2_GPU_CASES[name]
    lens = wl.draw_seq_lens(cfg)
    if cap < 0:
        probe = mb.Session(mb_config(cfg, lens))
        cap = -cap * probe.layout.weight_slot_bytes * cfg.R / probe.layout.resident_bytes
        probe.close()
    st, sess = gpu_session(cfg, lens, cap_frac=cap, fill="normal" if cfg.w_dtype == "fp8_e4m3_b128" else "tag",
                           initial_mode=first)
    assert sess.layout.w_shift_slots < (2 if cfg.w_orient else 1) and sess.layout.w_staging_bytes > 0
    owner, bt, _ = start(st, sess, first, "random")
    mode = first
    waves = 0
    for _ in range(3):
        mode, owner, bt, stats = gpu_switch(st, sess, mode, owner, bt)
        waves = max(waves, stats["n_w_waves"])
    assert waves > 0
    sess.close()


def shares_execute(bounds):
    def run(sess, plan):
        stream = torch.cuda.current_stream().cuda_stream
        mb.moebius_reshard_shares(sess.ctx, plan, bounds, 0, len(bounds) - 1, stream)
        mb.moebius_reshard_publish(sess.ctx, plan, stream)
    return run


BARRIER_CASES = {
    "smallish_2": (SMALLISH, [0, 2, 4], None, 0.0),
    "smallish_4": (SMALLISH, [0, 1, 2, 3, 4], None, 0.0),
    "uneven_3": (SMALLISH, [0, 1, 3, 4], None, 0.0),
    "tight_rounds_2": (SMALLISH.with_(L=1, n_req=40, seed=99), [0, 2, 4], "tight", 0.5),
    "replicated_heads_8": (wl.get_config("tiny").with_(R=8, E=8, I=64, kv_heads=4, n_req=7, len_dist=("uniform", 1, 70), seed=13),
                           list(range(9)), None, 0.0),
    "fp8_2": (wl.get_config("fp8_graph").with_(L=1, E=8, H=256, I=1536, n_req=6, len_dist=("uniform", 1, 60), seed=3),
              [0, 4, 8], None, 0.0),
    "inplace_waves_2": (SMALLISH.with_(w_inplace=1, seed=81), [0, 2, 4], None, 0.0),
    "attn_gather_2": (wl.get_config("tiny").with_(R=4, E=8, H=128, I=128, kv_heads=2, head_dim=32, n_q_heads=8, attn_mode=2, L=2,
                                                  n_req=9, len_dist=("uniform", 1, 80), seed=64), [0, 2, 4], None, 0.0),
    "small_config_4": (wl.get_config("small"), [0, 1, 2, 3, 4], None, 0.0),
}


@pytest.mark.parametrize("name", sorted(BARRIER_CASES))
def test_device_side_round_barrier(name):
    """the whole switch as ONE launch with the cross-share barrier on the
    device -- per-share tickets, per-wave flags in the flag page inside each share's first rank region
    (st.release.sys / ld.acquire.sys), here verified as one cooperative launch whose CTA groups play the
    GPUs.  Same waves as the host-barrier path; bit-exact with the oracle, both directions, and a plain
    fused switch can follow on the same buffers."""
    cfg, bounds, policy, cap = BARRIER_CASES[name]
    lens = wl.draw_seq_lens(cfg)
    st, sess = gpu_session(cfg, lens, policy, cap, fill="normal" if cfg.w_dtype == "fp8_e4m3_b128" else "tag")
    owner, bt, _ = start(st, sess, TP, "random", seed=2)
    mode = TP
    for k in range(4):
        mode, owner, bt, stats = gpu_switch(st, sess, mode, owner, bt, execute=shares_execute(bounds) if k != 2 else None)
    sess.close()


def test_device_side_round_barrier_argument_checks():
    st, sess = gpu_session(SMALLISH.with_(L=1))
    owner, bt, _ = start(st, sess, TP, "random")
    plan = sess.plan(EP, st.lens, owner, bt, from_mode=TP)
    for bad in ([0, 2], [1, 4], [0, 2, 2, 4], [0, 3, 2, 4]):
        with pytest.raises(mb.MoebiusError):
            mb.moebius_reshard_shares(sess.ctx, plan, bad, 0, len(bad) - 1, 0)
    with pytest.raises(mb.MoebiusError):
        mb.moebius_reshard_shares(sess.ctx, plan, [0, 2, 4], 1, 2, 0)     # shares 1..2 of 2
    assert mb.moebius_active_mode(sess.ctx) == TP
    sess.close()


@pytest.mark.parametrize("which", ["smallish", "small", "fp8"])
@pytest.mark.parametrize("first", [TP, EP])
def test_banded_chain_on_device(which, first):
    """moebius_set_chain_bands(ctx, 1): links cut into 2 x 2 segments that wait for one half of their
    predecessor (no device-wide drain between links).  Off by default -- measured slower -- but kept
    correct: bit-exact with the oracle, both directions."""
    cfg = {"smallish": SMALLISH, "small": wl.get_config("small"),
           "fp8": wl.get_config("fp8_graph").with_(L=2, E=16, H=256, I=1536, n_req=6, len_dist=("uniform", 1, 60), seed=3)}[which]
    st, sess = gpu_session(cfg, fill="normal" if cfg.w_dtype == "fp8_e4m3_b128" else "tag", initial_mode=first)
    mb.moebius_set_chain_bands(sess.ctx, True)
    owner, bt, _ = start(st, sess, first, "random")
    mode = first
    for _ in range(3):
        mode, owner, bt, stats = gpu_switch(st, sess, mode, owner, bt)
    assert stats["n_segments"] >= 4 * 3 * cfg.L
    sess.close()
