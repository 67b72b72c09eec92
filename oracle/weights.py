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
    raise ValueError(kind)


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
    if kind in ("gate", "up"):
        return np.ascontiguousarray(S[:, :, lo:hi])
    if kind == "down":
        return np.ascontiguousarray(S[:, lo:hi, :])
    raise ValueError(kind)


def ep_scale_view(S: np.ndarray, r: int, R: int) -> np.ndarray:
    E = S.shape[0]
    n = E // R
    return np.ascontiguousarray(S[r * n:(r + 1) * n])
