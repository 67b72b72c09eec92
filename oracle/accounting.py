"""Byte accounting by enumeration of destination slices.  TEST INFRASTRUCTURE ONLY.

PAPER.md:35: a switch "moves only the owner-changed bytes"; "the 1/P of each object
whose destination is the sending rank itself is a local HBM write rather than an interconnect
transfer".  Reading A15: `moved` = bytes of destination slices whose destination rank differs
from their source rank (every replica counted); `relocated` = all destination bytes written;
`read` = unique source bytes read.
"""
from __future__ import annotations

from .kv import kv_heads_of_rank, tp_source_rank


def weight_bytes(R, L, E, H, I, elem_bytes, direction: str):
    """Enumerate (expert e, TP rank j) slices of one matrix; 3 matrices per layer, L layers.
    EP owner of expert e is e div (E/R); a slice has H*(I/R) elements for every matrix kind."""
    slice_bytes = H * (I // R) * elem_bytes
    moved = relocated = 0
    for e in range(E):
        q = e // (E // R)
        for j in range(R):
            src, dst = (q, j) if direction == "ep2tp" else (j, q)
            relocated += slice_bytes
            if src != dst:
                moved += slice_bytes
    f = 3 * L
    return {"moved": moved * f, "relocated": relocated * f, "read": relocated * f}


def kv_bytes(seq_lens, owner, R, L, Hkv, D, elem_bytes, direction: str):
    """Per token and per pool (K and V of each layer: 2L pools).  `owner` is the EP-side owner
    vector (source owner for ep2tp, new owner for tp2ep)."""
    head_bytes = D * elem_bytes
    moved = relocated = read = 0
    for i, n in enumerate(seq_lens):
        n = int(n)
        o = int(owner[i])
        if direction == "ep2tp":
            read += n * Hkv * head_bytes
            for j in range(R):
                b = n * len(kv_heads_of_rank(j, R, Hkv)) * head_bytes
                relocated += b
                if j != o:
                    moved += b
        else:
            for h in range(Hkv):
                s = tp_source_rank(h, o, R, Hkv)
                relocated += n * head_bytes
                read += n * head_bytes
                if s != o:
                    moved += n * head_bytes
    f = 2 * L
    return {"moved": moved * f, "relocated": relocated * f, "read": read * f}


def scale_bytes(R, L, E, H, I, direction: str, kinds=("gate", "up", "down")):
    """fp8 block scales (BASELINE.json config 5; SURVEY.md §8(c) "bytes moved ... (+ scales)";
    reading A13), by enumeration of (expert e, TP rank j, 128-block ib of the intermediate axis).

    One fp32 scale per 128x128 block: an (e, ib) pair stands for the H/128 scales of that block
    column (gate/up/w2: [E, H/128, I/128]) or block row (down: [E, I/128, H/128]); the stacked
    `w13` ([E, 2I/128, H/128]) has every ib twice, once in the gate half and once in the up half.
    TP shard j carries every block its I/R columns touch, so a block that straddles two shards is
    held by both (like a replicated KV head):
      ep2tp  every holder j of (e, ib) receives a copy from the EP owner q = e div (E/R): each copy
             is `relocated`, and `moved` when j != q; the source is read once per (e, ib).
      tp2ep  the EP owner q receives (e, ib) once, read from its LOWEST-rank holder (the rule of
             reading A5 applied to scales): `moved` when that holder != q.
    """
    from .weights import tp_scale_blocks
    per_block = (H // 128) * 4
    holders = {}
    for j in range(R):
        lo, hi = tp_scale_blocks(j, R, I)
        for ib in range(lo, hi):
            holders.setdefault(ib, []).append(j)
    assert sorted(holders) == list(range(I // 128))
    moved = relocated = read = 0
    for e in range(E):
        q = e // (E // R)
        for ib in range(I // 128):
            if direction == "ep2tp":
                read += per_block
                for j in holders[ib]:
                    relocated += per_block
                    if j != q:
                        moved += per_block
            else:
                src = min(holders[ib])
                read += per_block
                relocated += per_block
                if src != q:
                    moved += per_block
    f = L * sum(2 if k == "w13" else 1 for k in kinds)
    return {"moved": moved * f, "relocated": relocated * f, "read": read * f}
