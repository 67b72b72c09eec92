"""Request ownership, block tables and paged-KV pool images.  TEST INFRASTRUCTURE ONLY.

PAPER.md:116 (§3.2): "Under EP ... each rank owns a disjoint subset of in-flight requests and
stores their KV cache for every head. Under TP ... every rank serves every request but stores only
its slice of the KV heads. When a model has fewer KV heads than ranks, TP replicates each head
across a group of ranks. For example, Qwen3's four KV heads at TP 8 place two ranks per head."
PAPER.md:122: paged blocks from a shared pool, tracked by a page table; target pages are
"reallocated under TP".  PAPER.md:124: TP->EP partition.  PAPER.md:126: nothing is dropped.
"""
from __future__ import annotations

import numpy as np


class CapacityError(Exception):
    """Target mode cannot hold the live requests (cancel the switch)."""


def kv_heads_of_rank(r: int, R: int, Hkv: int):
    """KV heads held by rank r under TP.  Hkv >= R: the r-th contiguous block of Hkv/R heads.
    Hkv < R: R/Hkv consecutive ranks per head, rank r holds head r div (R/Hkv) (reading A4)."""
    if Hkv >= R:
        if Hkv % R:
            raise ValueError("kv_heads % R != 0")
        hpr = Hkv // R
        return list(range(r * hpr, (r + 1) * hpr))
    if R % Hkv:
        raise ValueError("R % kv_heads != 0")
    return [r // (R // Hkv)]


def tp_source_rank(head: int, new_owner: int, R: int, Hkv: int) -> int:
    """TP->EP: which TP rank's copy of `head` is read for a request going to `new_owner`
    (reading A5): the new owner itself if it holds the head, else the lowest-rank holder."""
    if head in kv_heads_of_rank(new_owner, R, Hkv):
        return new_owner
    for j in range(R):
        if head in kv_heads_of_rank(j, R, Hkv):
            return j
    raise AssertionError


def _kv_dtype(KV):
    vals = list(KV.values()) if isinstance(KV, dict) else list(KV)
    return vals[0].dtype if vals else np.uint16   # no live request: an empty bf16 pool


def pages_needed(length: int, pg: int) -> int:
    return (int(length) + pg - 1) // pg


def partition_requests(seq_lens, R: int):
    """TP->EP request partition: "sorts requests by decreasing sequence length and
    greedily places each request on the least-loaded rank, balancing request and token counts
    together. The heuristic is deterministic".  Reading A9: sort key (-len, id); least loaded =
    lexicographically smallest (tokens, requests, rank id)."""
    n = len(seq_lens)
    order = sorted(range(n), key=lambda i: (-int(seq_lens[i]), i))
    tokens = [0] * R
    reqs = [0] * R
    owner = np.full(n, -1, dtype=np.int32)
    for i in order:
        best = 0
        for r in range(1, R):
            if (tokens[r], reqs[r], r) < (tokens[best], reqs[best], best):
                best = r
        owner[i] = best
        tokens[best] += int(seq_lens[i])
        reqs[best] += 1
    return owner


def canonical_block_tables(seq_lens, owner, mode: str, n_pages: int, pg: int, max_pages: int):
    """Target block tables after a switch (reading A7; "reallocated").

    Requests in ascending id, each gets ceil(len/pg) consecutive pages.
      TP: one table shared by all ranks, pages bump UP from page 0.
      EP: per owning rank, pages bump DOWN from the last page: the k-th page handed out on a rank
          is n_pages - 1 - k.
    Raises CapacityError when a pool cannot hold them."""
    n = len(seq_lens)
    bt = np.full((n, max_pages), -1, dtype=np.int32)
    if mode == "tp":
        nxt = 0
        for i in range(n):
            k = pages_needed(seq_lens[i], pg)
            if k > max_pages or nxt + k > n_pages:
                raise CapacityError("TP pool")
            for b in range(k):
                bt[i, b] = nxt + b
            nxt += k
        return bt
    if mode == "ep":
        used = {}
        for i in range(n):
            r = int(owner[i])
            k = pages_needed(seq_lens[i], pg)
            u = used.get(r, 0)
            if k > max_pages or u + k > n_pages:
                raise CapacityError("EP pool of rank %d" % r)
            for b in range(k):
                bt[i, b] = n_pages - 1 - (u + b)
            used[r] = u + k
        return bt
    raise ValueError(mode)


def tp_pool_image(KV, seq_lens, bt, r: int, R: int, Hkv: int, D: int, pg: int, n_pages: int):
    """K (or V) pool of rank r under TP for one layer: [n_pages, pg, hpr, D] plus a validity mask
    [n_pages, pg].  Token t of request i sits at page bt[i][t div pg], slot t mod pg, and holds
    rank r's heads only; every rank uses the same table.  KV[i] is the logical [len_i, Hkv, D].
    Bytes outside the mask are unspecified (reading A10)."""
    heads = kv_heads_of_rank(r, R, Hkv)
    pool = np.zeros((n_pages, pg, len(heads), D), dtype=_kv_dtype(KV))
    mask = np.zeros((n_pages, pg), dtype=bool)
    for i in range(len(seq_lens)):
        n = int(seq_lens[i])
        for b in range(pages_needed(n, pg)):          # block b holds tokens [b*pg, min(n, (b+1)*pg))
            p = int(bt[i][b])
            k = min(pg, n - b * pg)
            assert 0 <= p < n_pages and not mask[p].any()
            pool[p, :k] = KV[i][b * pg:b * pg + k][:, heads, :]
            mask[p, :k] = True
    return pool, mask


def ep_pool_image(KV, seq_lens, owner, bt, r: int, Hkv: int, D: int, pg: int, n_pages: int):
    """K (or V) pool of rank r under EP for one layer: [n_pages, pg, Hkv, D] + mask; holds all
    heads of the requests rank r owns and nothing else."""
    pool = np.zeros((n_pages, pg, Hkv, D), dtype=_kv_dtype(KV))
    mask = np.zeros((n_pages, pg), dtype=bool)
    for i in range(len(seq_lens)):
        if int(owner[i]) != r:
            continue
        n = int(seq_lens[i])
        for b in range(pages_needed(n, pg)):
            p = int(bt[i][b])
            k = min(pg, n - b * pg)
            assert 0 <= p < n_pages and not mask[p].any()
            pool[p, :k] = KV[i][b * pg:b * pg + k]
            mask[p, :k] = True
    return pool, mask


def gather_request_from_tp(pools, bt_row, length: int, R: int, Hkv: int, D: int, pg: int):
    """Reassemble the logical [len, Hkv, D] of one request from the R TP pools (reachability,
    PAPER.md:126).  For a replicated head the lowest-rank holder is read; the caller checks the
    replicas agree."""
    out = np.zeros((length, Hkv, D), dtype=pools[0].dtype)
    for h in range(Hkv):
        j = next(j for j in range(R) if h in kv_heads_of_rank(j, R, Hkv))
        hl = kv_heads_of_rank(j, R, Hkv).index(h)
        for t in range(length):
            out[t, h] = pools[j][int(bt_row[t // pg]), t % pg, hl]
    return out


def gather_request_from_ep(pool, bt_row, length: int, pg: int):
    out = np.zeros((length,) + pool.shape[2:], dtype=pool.dtype)
    for t in range(length):
        out[t] = pool[int(bt_row[t // pg]), t % pg]
    return out
