"""Fixed-address proof: one CUDA graph per mode is captured
ONCE, before the first switch.  It reads the expert weights (and fp8 scales) and the KV pools through
baked-in pointers -- the fixed views `moebius_view` reports -- and finds the KV pages through the
published table buffer, also at a baked-in address.  After every switch the graph of the now-active
mode is replayed and its outputs are compared with what the oracle builds from the logical tensors:
a switch changes contents, never addresses ("graphs embed addresses").

BASELINE.json config 5 (fp8 + graph stress): 8 back-to-back alternating switches, a replay between
each, outputs bit-exact.  Here at a reduced shape (whole views are copied out and compared); the
full-size variant is in test_gpu_fullsize.py.
"""
import numpy as np
import pytest

import oracle
import workloads as wl
from harness import EP, TP, OracleLayout, State, expected_target, mb, mb_config, source_tables

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

KINDS = ("gate", "up", "down")


class ModeGraph:
    """Captured reader of one mode's views.  Nothing in here is re-created after capture."""

    def __init__(self, sess, cfg, mode, n_req, with_scales):
        self.sess, self.cfg, self.mode, self.n = sess, cfg, mode, n_req
        lay = sess.layout
        mp = sess.cfg.max_pages_per_request
        self.mp = mp
        tids = list(range(3)) + ([5, 6, 7] if with_scales else [])
        self.w_views = {(r, l, t): sess.view(mode, r, l, t) for r in range(cfg.R) for l in range(cfg.L) for t in tids}
        self.kv_views = {(r, l, k): sess.view(mode, r, l, 3 + k) for r in range(cfg.R) for l in range(cfg.L) for k in range(2)}
        self.ptrs = [v.data_ptr() for v in list(self.w_views.values()) + list(self.kv_views.values())]
        tables = sess.tables
        self.out_w, self.out_kv = {}, {}
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):      # warm-up outside capture (allocator, lazy init)
            tables[lay.tbl_bt_off:lay.tbl_bt_off + n_req * mp].clamp(min=0).long()
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph):
            self.hdr = tables[:16].clone()
            self.owner = tables[lay.tbl_owner_off:lay.tbl_owner_off + n_req].clone()
            self.lens = tables[lay.tbl_lens_off:lay.tbl_lens_off + n_req].clone()
            bt = tables[lay.tbl_bt_off:lay.tbl_bt_off + n_req * mp]
            self.bt = bt.clone()
            idx = bt.clamp(min=0).long()                       # the page ids are read at REPLAY time
            for k, v in self.w_views.items():
                self.out_w[k] = v.clone()                      # dense copy through the baked-in pointer
            for k, v in self.kv_views.items():
                self.out_kv[k] = v.index_select(0, idx)        # [n*mp, pg, heads, D] gathered through the tables

    def replay(self):
        self.graph.replay()
        torch.cuda.synchronize()

    def check(self, st: State, want_owner, want_bt):
        cfg, n, mp = self.cfg, self.n, self.mp
        now = [self.sess.view(self.mode, r, l, t).data_ptr() for (r, l, t) in self.w_views] + \
              [self.sess.view(self.mode, r, l, 3 + k).data_ptr() for (r, l, k) in self.kv_views]
        assert now == self.ptrs                                # addresses never move
        hdr = self.hdr.cpu().numpy()
        assert hdr[0] == self.mode and hdr[1] == n
        assert np.array_equal(self.bt.cpu().numpy().reshape(n, mp), want_bt)
        assert np.array_equal(self.lens.cpu().numpy(), st.lens)
        owner = self.owner.cpu().numpy()
        assert np.array_equal(owner, want_owner if self.mode == EP else np.full(n, -1, np.int32))
        ol = oracle.OracleLayout(st, None, 0, 0, self.mode, want_owner, want_bt)
        for (r, l, t), out in self.out_w.items():
            want = ol.weight_view(r, l, KINDS[t]) if t < 3 else ol.scale_view(r, l, KINDS[t - 5])
            got = out.cpu().numpy()
            assert np.array_equal(got.view(np.uint8).reshape(-1), np.ascontiguousarray(want).view(np.uint8).reshape(-1)), (r, l, t)
        # KV: every token of every request is reachable through the published tables
        pg = cfg.page
        for (r, l, k), out in self.out_kv.items():
            got = out.cpu().numpy().view(np.uint16).reshape(n, mp * pg, -1, cfg.head_dim)
            heads = list(range(cfg.kv_heads)) if self.mode == EP else oracle.kv_heads_of_rank(r, cfg.R, cfg.kv_heads)
            KV = st.kv(l, k)
            for i in range(n):
                if self.mode == EP and want_owner[i] != r:
                    continue
                ln = int(st.lens[i])
                assert np.array_equal(got[i, :ln], KV[i][:, heads, :]), (r, l, k, i)


def run_graph_stress(cfg, n_switches, first=TP):
    assert torch.cuda.is_available()
    st = State(cfg, fill="normal" if cfg.w_dtype == "fp8_e4m3_b128" else "tag")
    sess = mb.Session(mb_config(cfg, st.lens, None, 0.0), device="cuda:0", initial_mode=first)
    n = len(st.lens)
    fp8 = cfg.w_dtype == "fp8_e4m3_b128"
    graphs = {m: ModeGraph(sess, cfg, m, n, fp8) for m in (TP, EP)}      # captured before any switch
    owner, bt = source_tables(st, sess, first, "random")
    image = np.full(sess.layout.base_bytes, 0xA5, np.uint8)
    OracleLayout(st, sess, first, owner, bt).place(image)
    sess.base[:image.size].copy_(torch.from_numpy(image))
    mode = first
    for _ in range(n_switches):
        to = EP if mode == TP else TP
        plan = sess.plan(to, st.lens, owner, bt, from_mode=mode)
        sess.reshard(plan)
        graphs[to].replay()                                              # same stream order: after the switch
        want_owner, want_bt = expected_target(st, sess, to)
        graphs[to].check(st, want_owner, want_bt)
        sess.free_plan(plan)
        owner, bt, mode = (want_owner if to == EP else None), want_bt, to
    sess.close()


def test_fp8_graph_stress_reduced():
    """Config 5 shape cut down: fp8 e4m3 experts + fp32 128x128 block scales, 4 KV heads on 8 ranks
    (replicated heads), geometric-tail lengths; 8 back-to-back alternating switches."""
    cfg = wl.get_config("fp8_graph").with_(L=2, E=16, H=256, I=1536, n_req=24, len_dist=("geometric", 60, 300), seed=11)
    run_graph_stress(cfg, 8)


def test_bf16_graph_replay_from_ep():
    cfg = wl.get_config("small").with_(L=2, H=128, I=256, n_req=12, len_dist=("uniform", 1, 150), seed=21)
    run_graph_stress(cfg, 4, first=EP)


def test_switch_itself_inside_a_captured_graph():
    """the switch launch captured ONCE in a CUDA graph (moebius_reshard_staged:
    fixed grid, fixed copy sizes, plan-dependent counts read from the uploaded header) and replayed
    for six plans -- both directions, the first from random tables in a tight pool (dependency rounds +
    staging): the plans differ in segment count, unit count and descriptor offsets.  The reader graph of the new mode is
    replayed after each and compared with the oracle."""
    cfg = wl.get_config("small").with_(L=2, H=128, I=256, n_req=30, len_dist=("uniform", 1, 200), seed=23)
    st = State(cfg, fill="tag")
    sess = mb.Session(mb_config(cfg, st.lens, "tight", 0.5), device="cuda:0", initial_mode=TP)
    n = len(st.lens)
    readers = {m: ModeGraph(sess, cfg, m, n, False) for m in (TP, EP)}
    owner, bt = source_tables(st, sess, TP, "random")
    image = np.full(sess.layout.base_bytes, 0xA5, np.uint8)
    OracleLayout(st, sess, TP, owner, bt).place(image)
    sess.base[:image.size].copy_(torch.from_numpy(image))
    # stage the first plan, warm the launch up once outside capture, then capture
    mode = TP
    plan = sess.plan(EP, st.lens, owner, bt, from_mode=mode)
    first_stats = mb.moebius_plan_stats(plan).as_dict()
    sess.stage(plan)
    with pytest.raises(mb.MoebiusError):          # staging made EP the active mode: the same plan no longer applies
        sess.stage(plan)
    switch_graph = torch.cuda.CUDAGraph()
    torch.cuda.synchronize()
    with torch.cuda.graph(switch_graph):
        sess.reshard_staged(torch.cuda.current_stream())
    seen = set()
    for k in range(6):
        to = EP if mode == TP else TP
        if k > 0:
            plan = sess.plan(to, st.lens, owner, bt, from_mode=mode)
            sess.stage(plan)
        s = mb.moebius_plan_stats(plan).as_dict()
        seen.add((s["n_segments"], s["n_units"]))
        switch_graph.replay()
        readers[to].replay()
        want_owner, want_bt = expected_target(st, sess, to)
        readers[to].check(st, want_owner, want_bt)
        torch.cuda.synchronize()                  # uploads of this replay are done: the next plan may be staged
        sess.free_plan(plan)
        owner, bt, mode = (want_owner if to == EP else None), want_bt, to
    assert first_stats["n_kv_rounds"] > 1         # the first plan really needed rounds
    assert len(seen) >= 2                          # the replays executed plans of different size
    sess.close()


def test_graph_replay_with_aliased_views():
    """The fixed-address proof with the in-place weight path (w_inplace = 1: the EP and the TP view of an
    object alias the same bytes): the reader graphs captured once replay correctly
    after every switch."""
    cfg = wl.get_config("small").with_(L=2, H=128, I=256, n_req=12, len_dist=("uniform", 1, 150), seed=25, w_inplace=1)
    run_graph_stress(cfg, 4)


def test_captured_switch_with_in_place_waves():
    """moebius_reshard_staged inside a captured graph, replayed for plans of the in-place path (dozens of
    dependency waves, parked blocks): everything plan-dependent is read from the uploaded image."""
    cfg = wl.get_config("small").with_(L=2, H=128, I=256, n_req=20, len_dist=("uniform", 1, 200), seed=27, w_inplace=1)
    st = State(cfg, fill="tag")
    sess = mb.Session(mb_config(cfg, st.lens), device="cuda:0", initial_mode=TP)
    n = len(st.lens)
    readers = {m: ModeGraph(sess, cfg, m, n, False) for m in (TP, EP)}
    owner, bt = source_tables(st, sess, TP, "random")
    image = np.full(sess.layout.base_bytes, 0xA5, np.uint8)
    OracleLayout(st, sess, TP, owner, bt).place(image)
    sess.base[:image.size].copy_(torch.from_numpy(image))
    mode = TP
    plan = sess.plan(EP, st.lens, owner, bt, from_mode=mode)
    assert mb.moebius_plan_stats(plan).as_dict()["n_w_waves"] > 0
    sess.stage(plan)
    switch_graph = torch.cuda.CUDAGraph()
    torch.cuda.synchronize()
    with torch.cuda.graph(switch_graph):
        sess.reshard_staged(torch.cuda.current_stream())
    for k in range(4):
        to = EP if mode == TP else TP
        if k > 0:
            plan = sess.plan(to, st.lens, owner, bt, from_mode=mode)
            sess.stage(plan)
        switch_graph.replay()
        readers[to].replay()
        want_owner, want_bt = expected_target(st, sess, to)
        readers[to].check(st, want_owner, want_bt)
        torch.cuda.synchronize()
        sess.free_plan(plan)
        owner, bt, mode = (want_owner if to == EP else None), want_bt, to
    sess.close()
