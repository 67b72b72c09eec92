"""MoE FFN computed from each layout, for the equivalence the paper states.  TEST INFRASTRUCTURE.

PAPER.md:46: the transformation produces "outputs equivalent to those the destination layout
would produce"; SwiGLU MLP with gate and up projections and a down projection;
PAPER.md:17: TP "synchronizes partial results with ... All-Reduce" (a sum of rank partials), EP
routes each token to the rank owning its expert.

y[t] = sum_k p[t,k] * ( silu(x[t] @ gate[e]) * (x[t] @ up[e]) ) @ down[e],  e = topk[t,k]
gate, up: [E, H, I]; down: [E, I, H].  Arithmetic in the dtype of the inputs (fp32 in the test;
fp64 for the dense reference).
"""
from __future__ import annotations

import numpy as np


def silu(a):
    return a / (1.0 + np.exp(-a))


def route_top2(logits: np.ndarray):
    """Reading of SURVEY.md §8(c): softmax -> top-2 -> renormalise.  Both layouts share it."""
    z = logits - logits.max(axis=1, keepdims=True)
    p = np.exp(z)
    p /= p.sum(axis=1, keepdims=True)
    idx = np.argsort(-p, axis=1, kind="stable")[:, :2]
    w = np.take_along_axis(p, idx, axis=1)
    w = w / w.sum(axis=1, keepdims=True)
    return idx, w


def moe_ffn_dense(x, gate, up, down, idx, w):
    y = np.zeros((x.shape[0], down.shape[2]), dtype=x.dtype)
    for t in range(x.shape[0]):
        for k in range(idx.shape[1]):
            e = idx[t, k]
            a = silu(x[t] @ gate[e]) * (x[t] @ up[e])
            y[t] += w[t, k] * (a @ down[e])
    return y


def moe_ffn_tp(x, gate_tp, up_tp, down_tp, idx, w):
    """gate_tp[r]: [E,H,I/R], up_tp[r] likewise, down_tp[r]: [E,I/R,H]; y = sum over ranks of the
    partial each rank computes from its shards alone (the All-Reduce)."""
    R = len(gate_tp)
    y = np.zeros((x.shape[0], down_tp[0].shape[2]), dtype=x.dtype)
    for r in range(R):
        part = np.zeros_like(y)
        for t in range(x.shape[0]):
            for k in range(idx.shape[1]):
                e = idx[t, k]
                a = silu(x[t] @ gate_tp[r][e]) * (x[t] @ up_tp[r][e])
                part[t] += w[t, k] * (a @ down_tp[r][e])
        y += part
    return y


def moe_ffn_ep(x, gate_ep, up_ep, down_ep, idx, w):
    """gate_ep[r]: [E/R,H,I] etc.; the token goes to the rank owning expert e = idx, which holds
    it whole at local index e mod (E/R)."""
    R = len(gate_ep)
    n_loc = gate_ep[0].shape[0]
    y = np.zeros((x.shape[0], down_ep[0].shape[2]), dtype=x.dtype)
    for t in range(x.shape[0]):
        for k in range(idx.shape[1]):
            e = int(idx[t, k])
            r, el = e // n_loc, e % n_loc
            assert r < R
            a = silu(x[t] @ gate_ep[r][el]) * (x[t] @ up_ep[r][el])
            y[t] += w[t, k] * (a @ down_ep[r][el])
    return y


# ---- the same FFN from the paper's orientation (W13 [E,2I,H], W2 [E,H,I]) ----------
# Row i of W13[e] is output channel i of the gate projection (i < I) or of the up projection
# (i >= I); W2[e] maps the I intermediate channels back to H:  a = silu(W13g x) * (W13u x), y = W2 a.

def moe_ffn_dense_w13(x, W13, W2, idx, w):
    I = W13.shape[1] // 2
    y = np.zeros((x.shape[0], W2.shape[1]), dtype=x.dtype)
    for t in range(x.shape[0]):
        for k in range(idx.shape[1]):
            e = idx[t, k]
            h = W13[e] @ x[t]
            y[t] += w[t, k] * (W2[e] @ (silu(h[:I]) * h[I:]))
    return y


def moe_ffn_tp_w13(x, W13_tp, W2_tp, idx, w):
    """W13_tp[r]: [E, 2I/R, H] (gate block then up block, reading A2), W2_tp[r]: [E, H, I/R]; each
    rank computes a partial from its shards alone, the All-Reduce sums them."""
    y = np.zeros((x.shape[0], W2_tp[0].shape[1]), dtype=x.dtype)
    for r in range(len(W13_tp)):
        wloc = W13_tp[r].shape[1] // 2
        part = np.zeros_like(y)
        for t in range(x.shape[0]):
            for k in range(idx.shape[1]):
                e = idx[t, k]
                h = W13_tp[r][e] @ x[t]
                part[t] += w[t, k] * (W2_tp[r][e] @ (silu(h[:wloc]) * h[wloc:]))
        y += part
    return y


def moe_ffn_ep_w13(x, W13_ep, W2_ep, idx, w):
    """W13_ep[r]: [E/R, 2I, H], W2_ep[r]: [E/R, H, I]; the owner of expert e computes it whole."""
    n_loc = W13_ep[0].shape[0]
    I = W13_ep[0].shape[1] // 2
    y = np.zeros((x.shape[0], W2_ep[0].shape[1]), dtype=x.dtype)
    for t in range(x.shape[0]):
        for k in range(idx.shape[1]):
            e = int(idx[t, k])
            r, el = e // n_loc, e % n_loc
            h = W13_ep[r][el] @ x[t]
            y[t] += w[t, k] * (W2_ep[r][el] @ (silu(h[:I]) * h[I:]))
    return y
