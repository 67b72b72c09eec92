"""Pins for the paper-orientation views (oracle.tp_w13_view / tp_w2_view, w_orient = 1; PAPER.md:100,
:110, readings A1/A2) and the FFN written from that orientation.  No GPU.  Each pin is something
other than the function's own slicing: a hand-worked fixture, the per-element index formula by
brute force, the relation to the (independently pinned) BASELINE.json-orientation views through a
transpose, tiling invariants, a reshape/transpose reduction, and the FFN equivalence
with negative controls that separate reading A2 from the other reading of "(E, 2I/P, H)"."""
import json
import os

import numpy as np
import pytest

import oracle
import workloads as wl


def test_golden_paper_orientation(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "weights_paper_orient_R2_E2_H2_I4.json")))
    R, E, H, I = (g["inputs"][k] for k in "REHI")
    W13 = np.arange(E * 2 * I * H).reshape(E, 2 * I, H)
    W2 = np.arange(E * H * I).reshape(E, H, I)
    for r in range(R):
        assert oracle.tp_w13_view(W13, r, R).ravel().tolist() == g["expected"]["w13_tp"][r]
        assert oracle.ep_weight_view(W13, r, R).ravel().tolist() == g["expected"]["w13_ep"][r]
        assert oracle.tp_w2_view(W2, r, R).ravel().tolist() == g["expected"]["w2_tp"][r]
        assert oracle.ep_weight_view(W2, r, R).ravel().tolist() == g["expected"]["w2_ep"][r]
        assert np.array_equal(oracle.tp_weight_view(W13, "w13", r, R), oracle.tp_w13_view(W13, r, R))


def test_bruteforce_per_element_tiny():
    # W13_tp[j][e][p*w + c][h] = W13[e][p*I + j*w + c][h]   (p = 0 gate, 1 up; w = I/R)
    # W2_tp[j][e][h][c]        = W2[e][h][j*w + c]
    cfg = wl.get_config("tiny").with_(w_orient=1)
    R, E, H, I = cfg.R, cfg.E, cfg.H, cfg.I
    w = I // R
    W13 = wl.gen_logical_weight(cfg, 0, "w13", fill="tag")
    W2 = wl.gen_logical_weight(cfg, 0, "w2", fill="tag")
    assert W13.shape == (E, 2 * I, H) and W2.shape == (E, H, I)
    for j in range(R):
        a = oracle.tp_w13_view(W13, j, R)
        b = oracle.tp_w2_view(W2, j, R)
        assert a.shape == (E, 2 * w, H) and b.shape == (E, H, w)
        for e in range(E):
            for p in range(2):
                for c in range(w):
                    for h in range(H):
                        assert a[e, p * w + c, h] == W13[e, p * I + j * w + c, h]
            for h in range(H):
                for c in range(w):
                    assert b[e, h, c] == W2[e, h, j * w + c]


@pytest.mark.parametrize("name", ["tiny", "small"])
def test_relation_to_baseline_orientation(name):
    """W13[e] = [gate[e]^T ; up[e]^T], W2[e] = down[e]^T.  The TP shard of the paper orientation must
    then be the transposed TP shards of the BASELINE.json orientation (pinned in
    test_oracle_weights.py) -- two independent slicings agreeing through a transpose."""
    cfg = wl.get_config(name)
    R = cfg.R
    gate = wl.gen_logical_weight(cfg, 0, "gate", fill="tag")
    up = wl.gen_logical_weight(cfg, 0, "up", fill="tag")
    down = wl.gen_logical_weight(cfg, 0, "down", fill="tag")
    W13 = np.concatenate([gate.transpose(0, 2, 1), up.transpose(0, 2, 1)], axis=1)
    W2 = down.transpose(0, 2, 1)
    w = cfg.I // R
    for r in range(R):
        a = oracle.tp_w13_view(W13, r, R)
        assert np.array_equal(a[:, :w, :], oracle.tp_weight_view(gate, "gate", r, R).transpose(0, 2, 1))
        assert np.array_equal(a[:, w:, :], oracle.tp_weight_view(up, "up", r, R).transpose(0, 2, 1))
        assert np.array_equal(oracle.tp_w2_view(W2, r, R), oracle.tp_weight_view(down, "down", r, R).transpose(0, 2, 1))
        assert np.array_equal(oracle.ep_weight_view(W2, r, R), oracle.ep_weight_view(down, r, R).transpose(0, 2, 1))


@pytest.mark.parametrize("name", ["tiny", "small"])
def test_tiling_and_reshape_reduction(name):
    cfg = wl.get_config(name).with_(w_orient=1)
    R, E, H, I = cfg.R, cfg.E, cfg.H, cfg.I
    w = I // R
    W13 = wl.gen_logical_weight(cfg, 0, "w13", fill="tag")
    W2 = wl.gen_logical_weight(cfg, 0, "w2", fill="tag")
    t13 = [oracle.tp_w13_view(W13, r, R) for r in range(R)]
    t2 = [oracle.tp_w2_view(W2, r, R) for r in range(R)]
    e13 = [oracle.ep_weight_view(W13, r, R) for r in range(R)]
    e2 = [oracle.ep_weight_view(W2, r, R) for r in range(R)]
    assert all(v.flags["C_CONTIGUOUS"] for v in t13 + t2 + e13 + e2)
    # shards tile the logical tensors: gate halves side by side rebuild the gate block, etc.
    assert np.array_equal(np.concatenate([t[:, :w] for t in t13], axis=1), W13[:, :I])
    assert np.array_equal(np.concatenate([t[:, w:] for t in t13], axis=1), W13[:, I:])
    assert np.array_equal(np.concatenate(t2, axis=2), W2)
    assert np.array_equal(np.concatenate(e13, axis=0), W13)
    # the relayout as one reshape/transpose of the EP stack: W13 EP [q,e',p,j,w,H] -> TP [j,(q,e'),p,w,H]
    red13 = np.stack(e13).reshape(R, E // R, 2, R, w, H).transpose(3, 0, 1, 2, 4, 5).reshape(R, E, 2 * w, H)
    red2 = np.stack(e2).reshape(R, E // R, H, R, w).transpose(3, 0, 1, 2, 4).reshape(R, E, H, w)
    for r in range(R):
        assert np.array_equal(red13[r], t13[r]) and np.array_equal(red2[r], t2[r])
    # single copy: same bytes per rank in both modes
    assert all(a.nbytes == b.nbytes for a, b in zip(t13 + t2, e13 + e2))


def _setup():
    cfg = wl.get_config("tiny").with_(w_dtype="fp32", w_orient=1)
    rng = np.random.default_rng(cfg.seed)
    W13 = wl.gen_logical_weight(cfg, 0, "w13")
    W2 = wl.gen_logical_weight(cfg, 0, "w2")
    x = rng.normal(size=(8, cfg.H)).astype(np.float32)
    idx, w = oracle.route_top2(rng.normal(size=(8, cfg.E)).astype(np.float32))
    return cfg, W13, W2, x, idx, w


def _rel(a, b):
    return float(np.linalg.norm(a.astype(np.float64) - b.astype(np.float64)) / np.linalg.norm(b.astype(np.float64)))


def test_ffn_tp_equals_ep_paper_orientation():
    cfg, W13, W2, x, idx, w = _setup()
    R, I = cfg.R, cfg.I
    t13 = [oracle.tp_w13_view(W13, r, R) for r in range(R)]
    t2 = [oracle.tp_w2_view(W2, r, R) for r in range(R)]
    e13 = [oracle.ep_weight_view(W13, r, R) for r in range(R)]
    e2 = [oracle.ep_weight_view(W2, r, R) for r in range(R)]
    y_tp = oracle.moe_ffn_tp_w13(x, t13, t2, idx, w)
    y_ep = oracle.moe_ffn_ep_w13(x, e13, e2, idx, w)
    y_ref = oracle.moe_ffn_dense_w13(x.astype(np.float64), W13.astype(np.float64), W2.astype(np.float64), idx,
                                     w.astype(np.float64))
    assert _rel(y_tp, y_ep) <= 1e-5 and _rel(y_tp, y_ref) <= 1e-5 and _rel(y_ep, y_ref) <= 1e-5
    # the same network written in the BASELINE.json orientation (independent code path) agrees
    gate, up, down = (W13[:, :I].transpose(0, 2, 1), W13[:, I:].transpose(0, 2, 1), W2.transpose(0, 2, 1))
    y0 = oracle.moe_ffn_dense(x.astype(np.float64), gate.astype(np.float64), up.astype(np.float64),
                              down.astype(np.float64), idx, w.astype(np.float64))
    assert _rel(y_ref, y0) <= 1e-12


def test_ffn_rejects_the_other_reading_of_the_tp_shard():
    """Reading A2.  "(E, 2I/P, H)" could also mean rows [r*2I/P, (r+1)*2I/P) of the stack; then rank
    0 would hold gate rows only and no rank could apply SwiGLU to its own shard: the sum of rank
    partials no longer equals the FFN.  Also: W2 columns paired with the wrong rank are detected."""
    cfg, W13, W2, x, idx, w = _setup()
    R, I = cfg.R, cfg.I
    t2 = [oracle.tp_w2_view(W2, r, R) for r in range(R)]
    t13 = [oracle.tp_w13_view(W13, r, R) for r in range(R)]
    y = oracle.moe_ffn_tp_w13(x, t13, t2, idx, w)
    step = 2 * I // R
    contiguous = [np.ascontiguousarray(W13[:, r * step:(r + 1) * step]) for r in range(R)]
    assert _rel(oracle.moe_ffn_tp_w13(x, contiguous, t2, idx, w), y) > 1e-2
    assert _rel(oracle.moe_ffn_tp_w13(x, t13, t2[::-1], idx, w), y) > 1e-2
    # up block first instead of gate block first is detected (silu(a)*b != silu(b)*a)
    wloc = I // R
    swapped = [np.ascontiguousarray(np.concatenate([t[:, wloc:], t[:, :wloc]], axis=1)) for t in t13]
    assert _rel(oracle.moe_ffn_tp_w13(x, swapped, t2, idx, w), y) > 1e-3


def test_fp8_scale_views_paper_orientation():
    """Reading A13 carried over: dequantised TP shard == dequantised logical rows/columns, bit-equal."""
    cfg = wl.get_config("fp8_graph").with_(E=8, H=256, I=1536, w_orient=1)   # I/R = 192 straddles blocks
    R, E, H, I = cfg.R, cfg.E, cfg.H, cfg.I
    w_ = I // R
    rng = np.random.default_rng(6)
    W13q = rng.integers(-8, 8, size=(E, 2 * I, H)).astype(np.float32)
    S13 = wl.gen_logical_scale(cfg, 0, "w13")
    assert S13.shape == (E, 2 * I // 128, H // 128)
    deq = W13q * np.repeat(np.repeat(S13, 128, axis=1), 128, axis=2)
    W2q = rng.integers(-8, 8, size=(E, H, I)).astype(np.float32)
    S2 = wl.gen_logical_scale(cfg, 0, "w2")
    deq2 = W2q * np.repeat(np.repeat(S2, 128, axis=1), 128, axis=2)
    for r in range(R):
        lo, hi = oracle.tp_scale_blocks(r, R, I)
        nb = hi - lo
        sv = oracle.tp_scale_view(S13, "w13", r, R, I)
        assert sv.shape == (E, 2 * nb, H // 128)
        wv = oracle.tp_w13_view(W13q, r, R)
        rows = (np.arange(r * w_, (r + 1) * w_) // 128) - lo          # block of each shard row, relative
        sc = np.concatenate([np.repeat(sv[:, :nb], 128, axis=2)[:, rows], np.repeat(sv[:, nb:], 128, axis=2)[:, rows]], axis=1)
        want = np.concatenate([deq[:, r * w_:(r + 1) * w_], deq[:, I + r * w_:I + (r + 1) * w_]], axis=1)
        assert np.array_equal((wv * sc).view(np.uint32), want.view(np.uint32))
        sv2 = oracle.tp_scale_view(S2, "w2", r, R, I)
        sc2 = np.repeat(sv2, 128, axis=1)[:, :, rows]
        assert np.array_equal((oracle.tp_w2_view(W2q, r, R) * sc2).view(np.uint32),
                              deq2[:, :, r * w_:(r + 1) * w_].view(np.uint32))
