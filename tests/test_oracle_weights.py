"""Pins for oracle/weights.py and oracle/ffn.py (no GPU).  Each pin is something other than the
oracle's own formula: hand-worked fixture, brute-force per-element index formula, concatenation
invariant, reshape/transpose reduction, and the FFN equivalence the paper states."""
import json
import os

import numpy as np
import pytest

import oracle
import workloads as wl


def test_golden_weights(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "weights_R2_E2_H2_I4.json")))
    R, E, H, I = (g["inputs"][k] for k in "REHI")
    gate = np.arange(E * H * I).reshape(E, H, I)
    down = np.arange(E * H * I).reshape(E, I, H)
    for r in range(R):
        assert oracle.tp_weight_view(gate, "gate", r, R).ravel().tolist() == g["expected"]["gate_tp"][r]
        assert oracle.tp_weight_view(gate, "up", r, R).ravel().tolist() == g["expected"]["gate_tp"][r]
        assert oracle.ep_weight_view(gate, r, R).ravel().tolist() == g["expected"]["gate_ep"][r]
        assert oracle.tp_weight_view(down, "down", r, R).ravel().tolist() == g["expected"]["down_tp"][r]
        assert oracle.ep_weight_view(down, r, R).ravel().tolist() == g["expected"]["down_ep"][r]


def test_bruteforce_per_element_tiny():
    # SURVEY.md §8(c) per-element form:
    #   gate_tp[j][e][h][c] = gate[e][h][j*I/R + c];  down_tp[j][e][c][h] = down[e][j*I/R + c][h]
    #   X_ep[q][e'][..] = X[q*E/R + e'][..]
    cfg = wl.get_config("tiny")
    R, E, H, I = cfg.R, cfg.E, cfg.H, cfg.I
    w = I // R
    gate = wl.gen_logical_weight(cfg, 0, "gate", fill="tag")
    down = wl.gen_logical_weight(cfg, 0, "down", fill="tag")
    for j in range(R):
        gt = oracle.tp_weight_view(gate, "gate", j, R)
        dt = oracle.tp_weight_view(down, "down", j, R)
        ge = oracle.ep_weight_view(gate, j, R)
        assert gt.shape == (E, H, w) and dt.shape == (E, w, H) and ge.shape == (E // R, H, I)
        for e in range(E):
            for h in range(H):
                for c in range(w):
                    assert gt[e, h, c] == gate[e, h, j * w + c]
                    assert dt[e, c, h] == down[e, j * w + c, h]
        for el in range(E // R):
            for h in range(H):
                for i in range(I):
                    assert ge[el, h, i] == gate[j * (E // R) + el, h, i]


@pytest.mark.parametrize("name", ["tiny", "small"])
def test_concat_and_reshape_reduction(name):
    cfg = wl.get_config(name)
    R, E, H, I = cfg.R, cfg.E, cfg.H, cfg.I
    for kind in ("gate", "up", "down"):
        X = wl.gen_logical_weight(cfg, 0, kind, fill="tag")
        tp = [oracle.tp_weight_view(X, kind, r, R) for r in range(R)]
        ep = [oracle.ep_weight_view(X, r, R) for r in range(R)]
        assert all(v.flags["C_CONTIGUOUS"] for v in tp + ep)
        # (iii) shards tile the logical tensor
        assert np.array_equal(np.concatenate(tp, axis=2 if kind != "down" else 1), X)
        assert np.array_equal(np.concatenate(ep, axis=0), X)
        # (i) the relayout as one reshape/transpose of the EP stack (SURVEY.md §7 structural fact)
        ep_stack = np.stack(ep)  # [q, e', ., .]
        if kind != "down":
            red = ep_stack.reshape(R, E // R, H, R, I // R).transpose(3, 0, 1, 2, 4).reshape(R, E, H, I // R)
        else:
            red = ep_stack.reshape(R, E // R, R, I // R, H).transpose(2, 0, 1, 3, 4).reshape(R, E, I // R, H)
        for r in range(R):
            assert np.array_equal(red[r], tp[r])
        # same byte count per rank in both modes (single copy)
        assert all(t.nbytes == e.nbytes for t, e in zip(tp, ep))


def test_special_cases():
    X = np.arange(4 * 2 * 4).reshape(4, 2, 4)
    # R = 1: both views are the logical tensor
    assert np.array_equal(oracle.tp_weight_view(X, "gate", 0, 1), X)
    assert np.array_equal(oracle.ep_weight_view(X, 0, 1), X)
    # E = R: one whole expert per rank
    assert np.array_equal(oracle.ep_weight_view(X, 2, 4), X[2:3])
    with pytest.raises(ValueError):
        oracle.tp_weight_view(X, "gate", 0, 3)


def _ffn_setup():
    cfg = wl.get_config("tiny").with_(w_dtype="fp32")
    rng = np.random.default_rng(cfg.seed)
    gate = wl.gen_logical_weight(cfg, 0, "gate")
    up = wl.gen_logical_weight(cfg, 0, "up")
    down = wl.gen_logical_weight(cfg, 0, "down")
    x = rng.normal(size=(8, cfg.H)).astype(np.float32)
    idx, w = oracle.route_top2(rng.normal(size=(8, cfg.E)).astype(np.float32))
    return cfg, gate, up, down, x, idx, w


def _rel(a, b):
    return float(np.linalg.norm(a.astype(np.float64) - b.astype(np.float64)) / np.linalg.norm(b.astype(np.float64)))


def test_ffn_tp_equals_ep_tiny_fp32():
    """PAPER.md:46 / BASELINE.json: TP-layout FFN (sum of rank partials) == EP-layout FFN, <= 1e-5."""
    cfg, gate, up, down, x, idx, w = _ffn_setup()
    R = cfg.R
    tp = [[oracle.tp_weight_view(X, k, r, R) for r in range(R)] for X, k in ((gate, "gate"), (up, "up"), (down, "down"))]
    ep = [[oracle.ep_weight_view(X, r, R) for r in range(R)] for X in (gate, up, down)]
    y_tp = oracle.moe_ffn_tp(x, *tp, idx, w)
    y_ep = oracle.moe_ffn_ep(x, *ep, idx, w)
    y_ref = oracle.moe_ffn_dense(x.astype(np.float64), gate.astype(np.float64), up.astype(np.float64),
                                 down.astype(np.float64), idx, w.astype(np.float64))
    assert y_tp.dtype == np.float32 and y_ep.dtype == np.float32
    assert _rel(y_tp, y_ep) <= 1e-5
    assert _rel(y_tp, y_ref) <= 1e-5 and _rel(y_ep, y_ref) <= 1e-5
    # routing sanity: two distinct experts, weights renormalised
    assert np.all(idx[:, 0] != idx[:, 1]) and np.allclose(w.sum(1), 1.0)


def test_ffn_detects_wrong_layouts():
    """Negative controls: plausible mistakes in the views break the equivalence."""
    cfg, gate, up, down, x, idx, w = _ffn_setup()
    R = cfg.R
    g = [oracle.tp_weight_view(gate, "gate", r, R) for r in range(R)]
    u = [oracle.tp_weight_view(up, "up", r, R) for r in range(R)]
    d = [oracle.tp_weight_view(down, "down", r, R) for r in range(R)]
    y = oracle.moe_ffn_tp(x, g, u, d, idx, w)
    # down shards paired with the wrong rank
    assert _rel(oracle.moe_ffn_tp(x, g, u, d[::-1], idx, w), y) > 1e-2
    # EP shards in the wrong owner order
    ep = [[oracle.ep_weight_view(X, r, R) for r in range(R)] for X in (gate, up, down)]
    assert _rel(oracle.moe_ffn_ep(x, ep[0][::-1], ep[1][::-1], ep[2][::-1], idx, w), y) > 1e-2
    # gate and up swapped is NOT detected by symmetry of silu? it is: silu(a)*b != silu(b)*a
    assert _rel(oracle.moe_ffn_tp(x, u, g, d, idx, w), y) > 1e-3


def test_fp8_scale_views():
    """Reading A13 pin: dequantised TP shard == dequantised logical slice, bit-equal in fp32."""
    cfg = wl.get_config("fp8_graph").with_(E=8, H=256, I=1536)  # I/R = 192: shards straddle blocks
    R, E, H, I = cfg.R, cfg.E, cfg.H, cfg.I
    rng = np.random.default_rng(5)
    for kind in ("gate", "down"):
        shape = (E, H, I) if kind == "gate" else (E, I, H)
        Wq = rng.integers(-8, 8, size=shape).astype(np.float32)  # stand-in for decoded e4m3 codes
        S = wl.gen_logical_scale(cfg, 0, kind)
        ax_i = 2 if kind == "gate" else 1
        # logical dequant: scale of block (h//128, i//128)
        Sfull = np.repeat(np.repeat(S, 128, axis=1), 128, axis=2)
        deq = Wq * Sfull
        for r in range(R):
            lo, hi = oracle.tp_scale_blocks(r, R, I)
            assert hi - lo == 2  # 192-wide shard always touches 2 blocks at this shape
            sv = oracle.tp_scale_view(S, kind, r, R, I)
            wv = oracle.tp_weight_view(Wq, kind, r, R)
            w_ = I // R
            # dequantise the shard with ITS OWN scale view: block index relative to lo
            cols = (np.arange(r * w_, (r + 1) * w_) // 128) - lo
            if kind == "gate":
                sc = np.repeat(sv, 128, axis=1)[:, :, cols]
            else:
                sc = np.repeat(sv, 128, axis=2)[:, cols, :]
            got = wv * sc
            want = np.take(deq, np.arange(r * w_, (r + 1) * w_), axis=ax_i)
            assert np.array_equal(got.view(np.uint32), want.view(np.uint32))
        ev = [oracle.ep_scale_view(S, r, R) for r in range(R)]
        assert np.array_equal(np.concatenate(ev, 0), S)
    # aligned case: no duplication
    assert oracle.tp_scale_blocks(1, 4, 512) == (1, 2)
