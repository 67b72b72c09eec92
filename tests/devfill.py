"""Test-only: fill the DEVICE with the TP-mode source state of a full-size workload, using torch ops.

At the Qwen3-235B shape the state is ~143 GB: it cannot be built on the host and uploaded the way
the small parity tests do.  Instead every element is written on the device as the tag value of its
LOGICAL coordinate (`workloads.tag_fill_u16_torch`, the same counter-based generator as the numpy
`workloads.tag_fill_u16` behind `gen_logical_weight(fill="tag")` / `gen_kv_request(fill="tag")`).
The tests then regenerate the logical tensors of SAMPLED objects on the host with numpy, let the
oracle build their target-mode views, and compare those with what the device holds after the switch.
Nothing here is used by the product, and nothing here produces an expected value.
"""
from __future__ import annotations

import numpy as np
import torch

import workloads as wl

KINDS = ("gate", "up", "down")
TENSOR_ID = {"gate": 0, "up": 1, "down": 2, "w13": 8, "w2": 9}   # moebius_tensor_t


def fill_random(sess):
    """Every byte of the unified buffer random: stale bytes never look like the right ones."""
    n8 = sess.base.numel() // 8 * 8
    sess.base[:n8].view(torch.int64).random_()


def _store(view, vals):
    if view.dtype == torch.uint8:
        view.copy_((vals & 0xFF).to(torch.uint8))
    elif view.dtype == torch.int16:
        view.copy_(vals.to(torch.int16))          # wraps to the same 16 bits
    else:
        view.copy_(vals.to(torch.float32))


def fill_tp_weight(sess, cfg, layer, kind, experts_per_chunk=16):
    """TP views of one (layer, kind) object on every rank <- tag of the logical coordinate."""
    dev = sess.base.device
    R, E, H, I = cfg.R, cfg.E, cfg.H, cfg.I
    w = I // R
    off = wl.tag_salt_offset(wl.weight_tag_salt(cfg, layer, kind))
    tid = TENSOR_ID[kind]
    for j in range(R):
        view = sess.view(0, j, layer, tid)
        for e0 in range(0, E, experts_per_chunk):
            e = torch.arange(e0, min(E, e0 + experts_per_chunk), device=dev, dtype=torch.int64)
            h = torch.arange(H, device=dev, dtype=torch.int64)
            c = torch.arange(w, device=dev, dtype=torch.int64) + j * w
            if kind in ("gate", "up", "w2"):   # logical [E,H,I]; TP shard j = columns [j*w, (j+1)*w)
                flat = (e[:, None, None] * H + h[None, :, None]) * I + c[None, None, :]
            elif kind == "down":               # logical [E,I,H]; TP shard j = rows [j*w, (j+1)*w)
                flat = (e[:, None, None] * I + c[None, :, None]) * H + h[None, None, :]
            else:                              # w13: logical [E,2I,H]; TP shard j = gate rows [j*w, (j+1)*w) then
                c2 = torch.cat([c, c + I])     # the same rows of the up half (reading A2)
                flat = (e[:, None, None] * (2 * I) + c2[None, :, None]) * H + h[None, None, :]
            _store(view[e0:e0 + len(e)], wl.tag_fill_u16_torch(flat, off))
            del flat


def tp_heads_of_rank(r, R, Hkv):
    return list(range(r * (Hkv // R), (r + 1) * (Hkv // R))) if Hkv >= R else [r // (R // Hkv)]


def fill_tp_pool(sess, cfg, layer, kvi, lens, bt, tokens_per_chunk=1 << 18):
    """TP pools of one (layer, K|V) on every rank <- tag of (request, token, head, d), placed through
    the SOURCE block tables `bt` (shared by all ranks under TP)."""
    dev = sess.base.device
    R, Hkv, D, pg = cfg.R, cfg.kv_heads, cfg.head_dim, cfg.page
    lens = np.asarray(lens, np.int64)
    req = np.repeat(np.arange(len(lens), dtype=np.int64), lens)
    tok = np.concatenate([np.arange(n, dtype=np.int64) for n in lens]) if len(lens) else np.zeros(0, np.int64)
    row = np.asarray(bt, np.int64)[req, tok // pg] * pg + tok % pg          # pool row (page*pg + slot) of every token
    offs = np.array([wl.tag_salt_offset(wl.kv_tag_salt(cfg, layer, kvi, i)) for i in range(len(lens))], np.int64)
    d = torch.arange(D, device=dev, dtype=torch.int64)
    for r in range(R):
        heads = torch.tensor(tp_heads_of_rank(r, R, Hkv), device=dev, dtype=torch.int64)
        pool = sess.view(0, r, layer, 3 + kvi)
        rows = pool.view(pool.shape[0] * pg, pool.shape[2], D)
        for a in range(0, len(req), tokens_per_chunk):
            b = min(len(req), a + tokens_per_chunk)
            t = torch.from_numpy(tok[a:b]).to(dev)
            o = torch.from_numpy(offs[req[a:b]]).to(dev)
            flat = (t[:, None, None] * Hkv + heads[None, :, None]) * D + d[None, None, :]
            vals = wl.tag_fill_u16_torch(flat, o[:, None, None])
            rows[torch.from_numpy(row[a:b]).to(dev)] = vals.to(torch.int16)


def weighted_checksum(view):
    """Two int64 checksums of a device view: the plain sum of its 16-bit (or 8-bit) words and a
    position-weighted sum.  The first is invariant under any permutation of the elements, the
    second only under the identity."""
    x = view.reshape(-1).to(torch.int64)
    n = x.numel()
    pos = torch.arange(n, device=x.device, dtype=torch.int64) % 65521 + 1
    return int(x.sum()), int((x * pos).sum())
