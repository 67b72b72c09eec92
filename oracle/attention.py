"""Attention-weight layouts of the two modes.  TEST INFRASTRUCTURE ONLY.

PAPER.md:112 (section 3.1): "Under EP, attention is data-parallel and every rank holds the full query,
key, value, and output projections.  Under TP, attention is tensor-parallel and each rank holds only
its head shard.  By default, Moebius keeps both layouts resident and switches attention weights by
pointer swap, paying one duplicated head shard per rank.  A memory-saving variant keeps only the
active layout and rebuilds TP-EP with an All-Gather."
PAPER.md:411 (App. C): "1.7 GB of TP-mode qkv_proj and o_proj shards held alongside the full EP
copies"; "64 heads of dimension 128, so its q/k/v/o projections total roughly 13 GB in BF16 across
its 94 layers.  TP holds one-eighth per GPU, EP a full copy".

Logical tensors of one layer (the paper fixes no storage orientation; reading A19):
    wq [Hq,  D, H]   query projection, one [D, H] block per query head
    wk [Hkv, D, H]   key projection            wv [Hkv, D, H]   value projection
    wo [H, Hq, D]    output projection: column block (head h) multiplies head h's output
EP view of every rank = the whole tensor.  TP view of rank r = its HEAD SHARD: query heads
[r*Hq/R, (r+1)*Hq/R) of wq and the same heads' columns of wo; KV heads exactly as the KV cache places
them (reading A4: kv_heads_of_rank) for wk and wv -- so a rank's query heads always find
their KV head on the same rank (grouped-query attention: query head h uses KV head h div (Hq/Hkv)).
"""
from __future__ import annotations

import numpy as np

from .kv import kv_heads_of_rank

ATTN_KINDS = ("wq", "wk", "wv", "wo")


def attn_shape(kind: str, Hq: int, Hkv: int, D: int, H: int):
    return {"wq": (Hq, D, H), "wk": (Hkv, D, H), "wv": (Hkv, D, H), "wo": (H, Hq, D)}[kind]


def q_heads_of_rank(r: int, R: int, Hq: int):
    """Query heads of rank r under TP: the r-th contiguous block of Hq/R heads."""
    if Hq % R:
        raise ValueError("n_q_heads % R != 0")
    w = Hq // R
    return list(range(r * w, (r + 1) * w))


def attn_ep_view(X: np.ndarray, r: int, R: int) -> np.ndarray:
    """EP: data-parallel attention, every rank holds the full projection."""
    return np.ascontiguousarray(X)


def attn_tp_view(X: np.ndarray, kind: str, r: int, R: int, Hq: int, Hkv: int) -> np.ndarray:
    """TP: rank r's head shard.  wq -> [Hq/R, D, H]; wk, wv -> [hpr, D, H] with the
    rank's KV heads (replicated when Hkv < R); wo -> [H, Hq/R, D]."""
    if kind == "wq":
        return np.ascontiguousarray(X[q_heads_of_rank(r, R, Hq)])
    if kind in ("wk", "wv"):
        return np.ascontiguousarray(X[kv_heads_of_rank(r, R, Hkv)])
    if kind == "wo":
        return np.ascontiguousarray(X[:, q_heads_of_rank(r, R, Hq), :])
    raise ValueError(kind)


# ---- what the layouts must compute (pins) ----------------------------------------------------------

def _softmax(a):
    a = a - a.max(axis=-1, keepdims=True)
    e = np.exp(a)
    return e / e.sum(axis=-1, keepdims=True)


def _heads_forward(x, wq_h, wk_h, wv_h, wo_h, kv_of_q):
    """Causal-free attention of a block of query heads over the tokens of x [T, H] (one sequence):
    wq_h [nq, D, H], wk_h/wv_h [nkv, D, H], wo_h [H, nq, D]; kv_of_q[i] = index into wk_h of query
    head i's KV head.  Returns this block's contribution to the output projection, [T, H]."""
    T = x.shape[0]
    D = wq_h.shape[1]
    y = np.zeros((T, wo_h.shape[0]), dtype=x.dtype)
    for i in range(wq_h.shape[0]):
        q = x @ wq_h[i].T                       # [T, D]
        k = x @ wk_h[kv_of_q[i]].T
        v = x @ wv_h[kv_of_q[i]].T
        p = _softmax((q @ k.T) / np.sqrt(D).astype(x.dtype))
        y += (p @ v) @ wo_h[:, i, :].T           # [T, D] @ [D, H]
    return y


def attn_forward_dense(x, wq, wk, wv, wo):
    """The model's attention block from the logical tensors (grouped-query attention)."""
    Hq, Hkv = wq.shape[0], wk.shape[0]
    g = Hq // Hkv
    return _heads_forward(x, wq, wk, wv, wo, [h // g for h in range(Hq)])


def attn_forward_tp(x, views, R, Hq, Hkv):
    """Tensor-parallel attention: rank r computes its heads from ITS OWN views only
    (views[r] = {"wq","wk","wv","wo"} TP views) and the All-Reduce sums the partial outputs."""
    g = Hq // Hkv
    y = None
    for r in range(R):
        kv_heads = kv_heads_of_rank(r, R, Hkv)
        kv_of_q = []
        for h in q_heads_of_rank(r, R, Hq):
            kv_of_q.append(kv_heads.index(h // g))      # raises if the rank lacks the KV head it needs
        part = _heads_forward(x, views[r]["wq"], views[r]["wk"], views[r]["wv"], views[r]["wo"], kv_of_q)
        y = part if y is None else y + part
    return y


def attn_forward_ep(x, view):
    """Data-parallel attention on one rank from its full copy."""
    return attn_forward_dense(x, view["wq"], view["wk"], view["wv"], view["wo"])


# ---- byte accounting (readings A15, A19) -----------------------------------------

def attn_bytes(R, L, Hq, Hkv, D, H, elem_bytes, direction: str, variant: str):
    """By enumeration of (tensor, head, destination rank).
    variant "dual"   (the paper's default): both layouts resident, the switch is a pointer swap --
                     nothing moves; `duplicated_per_rank` = the TP head shard held beside the full copy.
    variant "gather" (the memory-saving variant): only the active layout is valid.  TP->EP rebuilds the
                     full projections on every rank from the R head shards (an All-Gather): rank q
                     receives every head it does not hold; a head it holds itself stays where it is
                     (reading A19: the TP shard is that head's own place inside the full tensor).  Source
                     of a replicated KV head: the lowest-rank holder (the rule of reading A5).
                     EP->TP keeps the local slice: nothing moves."""
    head = D * H * elem_bytes                   # one head's block of any of the four projections
    shard = full = 0
    moved = relocated = read = 0
    for r in range(R):
        nq, nkv = len(q_heads_of_rank(r, R, Hq)), len(kv_heads_of_rank(r, R, Hkv))
        if r == 0:
            shard = (2 * nq + 2 * nkv) * head      # wq + wo shards, wk + wv shards
            full = (2 * Hq + 2 * Hkv) * head
        if variant == "gather" and direction == "tp2ep":
            for kind, heads_of in (("wq", lambda j: q_heads_of_rank(j, R, Hq)), ("wo", lambda j: q_heads_of_rank(j, R, Hq)),
                                   ("wk", lambda j: kv_heads_of_rank(j, R, Hkv)), ("wv", lambda j: kv_heads_of_rank(j, R, Hkv))):
                n_heads = Hq if kind in ("wq", "wo") else Hkv
                for h in range(n_heads):
                    if h in heads_of(r):
                        continue                    # already in place on rank r
                    src = min(j for j in range(R) if h in heads_of(j))
                    assert src != r
                    relocated += head
                    moved += head
                    read += head
    return {"moved": moved * L, "relocated": relocated * L, "read": read * L,
            "duplicated_per_rank": shard * L if variant == "dual" else 0,
            "full_per_rank": full * L, "shard_per_rank": shard * L}
