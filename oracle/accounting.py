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
