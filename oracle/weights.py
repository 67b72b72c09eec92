"""Expert-weight layouts, written out as the paper defines them.  TEST INFRASTRUCTURE ONLY.

PAPER.md:100 (§3.1): "Under EP, each rank owns a disjoint subset of complete experts. It owns
E_local = E/P experts ...  Under TP, each rank owns one shard of every expert".
PAPER.md:110: "The gate-up and down projections reshard symmetrically, along the output and
input intermediate dimensions, respectively."

Orientation (reading A1, BASELINE.json): gate, up are separate logical tensors [E, H, I] (the
intermediate dimension is the LAST axis), down is [E, I, H] (intermediate is the MIDDLE axis).
So a TP shard of gate/up is a block of I/R columns, a TP shard of down the matching I/R rows.
Rank r's shard is the r-th contiguous block (BASELINE.json north_star: "columns
[r*I/R,(r+1)*I/R) of every expert's gate/up and the matching rows of down").
"""
from __future__ import annotations

import numpy as np


def _check(E, I, R):
    if E % R or I % R:
        raise ValueError("E and I must be divisible by R (reading A3)")


def tp_weight_view(X: np.ndarray, kind: str, r: int, R: int) -> np.ndarray:
    """Dense TP view of rank r.  gate/up: [E, H, I/R]; down: [E, I/R, H].  Experts in global order."""
    if kind in ("gate", "up"):
        E, H, I = X.shape
        _check(E, I, R)
        w = I // R
        return np.ascontiguousarray(X[:, :, r * w:(r + 1) * w])
    if kind == "down":
        E, I, H = X.shape
        _check(E, I, R)
        w = I // R
        return np.ascontiguousarray(X[:, r * w:(r + 1) * w, :])
    if kind == "w13":
        return tp_w13_view(X, r, R)
    if kind == "w2":
        return tp_w2_view(X, r, R)
    raise ValueError(kind)


# ---- the paper's own orientation (readings A1/A2; w_orient = 1) --------------------
# "stores the full gate-up projection W13 with shape (E_local, 2I, H), where the leading factor of
# two stacks the gate and up projections of the SwiGLU MLP, and the full down projection W2 with
# shape (E_local, H, I).  Under TP ... W13 has shape (E, 2I/P, H), and W2 has shape (E, H, I/P)."
# gate-up reshards along the OUTPUT intermediate dimension (rows of W13), down along
# the INPUT intermediate dimension (columns of W2).

def tp_w13_view(W13: np.ndarray, r: int, R: int) -> np.ndarray:
    """[E, 2I, H] -> [E, 2I/R, H].  Reading A2 (per projection): rank r takes rows
    [r*I/R, (r+1)*I/R) of the gate half (rows 0..I-1) and the same rows of the up half
    (rows I..2I-1), gate block first -- so every rank can run SwiGLU on its own shard."""
    E, I2, H = W13.shape
    if I2 % 2:
        raise ValueError("W13 stacks gate and up: its middle axis must be even")
    I = I2 // 2
    _check(E, I, R)
    w = I // R
    gate_rows = W13[:, r * w:(r + 1) * w, :]
    up_rows = W13[:, I + r * w:I + (r + 1) * w, :]
    return np.ascontiguousarray(np.concatenate([gate_rows, up_rows], axis=1))


def tp_w2_view(W2: np.ndarray, r: int, R: int) -> np.ndarray:
    """[E, H, I] -> [E, H, I/R]: columns [r*I/R, (r+1)*I/R) (the input-intermediate dimension)."""
    E, H, I = W2.shape
    _check(E, I, R)
    w = I // R
    return np.ascontiguousarray(W2[:, :, r * w:(r + 1) * w])


def ep_weight_view(X: np.ndarray, r: int, R: int) -> np.ndarray:
    """Dense EP view of rank r: experts [r*E/R, (r+1)*E/R) whole (any kind)."""
    E = X.shape[0]
    if E % R:
        raise ValueError("E must be divisible by R")
    n = E // R
    return np.ascontiguousarray(X[r * n:(r + 1) * n])


# ---- fp8 per-128x128-block scales (not in the paper; BASELINE.json config 5, reading A13) -------

def tp_scale_blocks(r: int, R: int, I: int, block: int = 128):
    """Indices of the 128-wide blocks along the intermediate axis that TP shard r touches:
    floor(r*I/R / 128) ... floor(((r+1)*I/R - 1) / 128), inclusive.  A straddled block is carried
    by both neighbours (duplicated, like a replicated KV head)."""
    w = I // R
    lo = (r * w) // block
    hi = ((r + 1) * w - 1) // block
    return lo, hi + 1  # half-open


def tp_scale_view(S: np.ndarray, kind: str, r: int, R: int, I: int) -> np.ndarray:
    """gate/up scales [E, H/128, I/128] -> [E, H/128, nb_r]; down scales [E, I/128, H/128] ->
    [E, nb_r, H/128], nb_r = number of blocks shard r touches."""
    lo, hi = tp_scale_blocks(r, R, I)
    if kind in ("gate", "up", "w2"):      # w2 scales [E, H/128, I/128]: intermediate blocks last
        return np.ascontiguousarray(S[:, :, lo:hi])
    if kind == "down":
        return np.ascontiguousarray(S[:, lo:hi, :])
    if kind == "w13":
        # scales [E, 2I/128, H/128]: the shard carries the blocks its gate rows touch, then the
        # blocks its up rows touch (the same block indices, offset by I/128) -> [E, 2*nb_r, H/128]
        ib = I // 128
        return np.ascontiguousarray(np.concatenate([S[:, lo:hi, :], S[:, ib + lo:ib + hi, :]], axis=1))
    raise ValueError(kind)


def ep_scale_view(S: np.ndarray, r: int, R: int) -> np.ndarray:
    E = S.shape[0]
    n = E // R
    return np.ascontiguousarray(S[r * n:(r + 1) * n])
