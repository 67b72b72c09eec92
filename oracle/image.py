"""Placing oracle layouts into a byte image of the unified buffer, and comparing.  TEST INFRASTRUCTURE.

The oracle does not know the address map: the caller passes `view_fn(mode, rank, layer, tensor_id)
-> (byte_offset, shape, elem_bytes)` (the fixed views the library reports) and the
pool page counts.  Nothing here imports the CUDA path.  mode: 0 = TP, 1 = EP; tensor ids: 0 gate,
1 up, 2 down, 3 K pool, 4 V pool, 5/6/7 fp8 scales of gate/up/down; paper orientation (w_orient = 1,
PAPER.md:100): 8 W13, 9 W2, 10/11 their fp8 scales; attention projections: 12 wq, 13 wk,
14 wv, 15 wo.  A view description may carry a 4th item, its strides in elements (the TP view of wo in
the memory-saving variant sits in place inside the full tensor).
"""
from __future__ import annotations

import numpy as np

import workloads as wl

from . import attention as oat
from . import kv as okv
from . import weights as ow

KINDS = ("gate", "up", "down")
ATTN_IDS = {"wq": 12, "wk": 13, "wv": 14, "wo": 15}
TP, EP = 0, 1


def weight_tensors(cfg):
    """[(kind, tensor id, scale tensor id)] of the orientation the config names."""
    if getattr(cfg, "w_orient", 0) == 1:
        return [("w13", 8, 10), ("w2", 9, 11)]
    return [("gate", 0, 5), ("up", 1, 6), ("down", 2, 7)]


class State:
    """Logical state of one workload: expert tensors per layer, K/V per request, lengths."""

    def __init__(self, cfg: wl.Config, seq_lens=None, fill="tag"):
        self.cfg = cfg
        self.lens = np.asarray(wl.draw_seq_lens(cfg) if seq_lens is None else seq_lens, dtype=np.int32)
        self.fill = fill
        self._w = {}
        self._kv = {}

    def weight(self, layer, kind):
        key = (layer, kind)
        if key not in self._w:
            self._w[key] = wl.gen_logical_weight(self.cfg, layer, kind, fill=self.fill)
        return self._w[key]

    def scale(self, layer, kind):
        return wl.gen_logical_scale(self.cfg, layer, kind)

    def attn(self, layer, kind):
        return wl.gen_attn_weight(self.cfg, layer, kind, fill=self.fill)

    def kv(self, layer, kvi):
        key = (layer, kvi)
        if key not in self._kv:
            self._kv[key] = {i: wl.gen_kv_request(self.cfg, layer, kvi, i, int(n), fill=self.fill)
                             for i, n in enumerate(self.lens)}
        return self._kv[key]

    def drop_cache(self):
        self._w.clear()
        self._kv.clear()


def np_view(image: np.ndarray, desc):
    off, shape, eb = desc[:3]
    dt = {1: np.uint8, 2: np.uint16, 4: np.float32}[eb]
    n = int(np.prod(shape)) * eb
    if len(desc) > 3 and desc[3] is not None:
        strides = tuple(desc[3])
        dense, st = [], 1
        for d in reversed(shape):
            dense.insert(0, st)
            st *= d
        if tuple(dense) != strides:        # a strided window onto the image (writable)
            span = (sum((d - 1) * s for d, s in zip(shape, strides)) + 1) * eb
            flat = image[off:off + span].view(dt)
            return np.lib.stride_tricks.as_strided(flat, shape=shape, strides=tuple(s * eb for s in strides))
    return image[off:off + n].view(dt).reshape(shape)


class OracleLayout:
    """The oracle's views of one mode for a State and a request state (owner, bt)."""

    def __init__(self, st: State, view_fn, pages_tp: int, pages_ep: int, mode: int, owner, bt):
        self.st, self.view_fn, self.mode, self.owner, self.bt = st, view_fn, mode, owner, bt
        self.pages_tp, self.pages_ep = pages_tp, pages_ep

    def weight_view(self, r, layer, kind):
        X = self.st.weight(layer, kind)
        R = self.st.cfg.R
        return ow.tp_weight_view(X, kind, r, R) if self.mode == TP else ow.ep_weight_view(X, r, R)

    def scale_view(self, r, layer, kind):
        S = self.st.scale(layer, kind)
        c = self.st.cfg
        return ow.tp_scale_view(S, kind, r, c.R, c.I) if self.mode == TP else ow.ep_scale_view(S, r, c.R)

    def attn_view(self, r, layer, kind, mode=None):
        c = self.st.cfg
        X = self.st.attn(layer, kind)
        if (self.mode if mode is None else mode) == TP:
            return oat.attn_tp_view(X, kind, r, c.R, c.n_q_heads, c.kv_heads)
        return oat.attn_ep_view(X, r, c.R)

    def attn_modes(self):
        """Which modes' attention views hold valid bytes while the buffer is in self.mode: both when both
        layouts are kept resident (attn_mode 1, PAPER.md:112 'pointer swap'), else the active one only."""
        m = getattr(self.st.cfg, "attn_mode", 0)
        return () if not m else ((TP, EP) if m == 1 else (self.mode,))

    def pool(self, r, layer, kvi):
        c = self.st.cfg
        KV = self.st.kv(layer, kvi)
        if self.mode == TP:
            return okv.tp_pool_image(KV, self.st.lens, self.bt, r, c.R, c.kv_heads, c.head_dim, c.page, self.pages_tp)
        return okv.ep_pool_image(KV, self.st.lens, self.owner, self.bt, r, c.kv_heads, c.head_dim, c.page,
                                 self.pages_ep)

    def place(self, image: np.ndarray):
        c = self.st.cfg
        fp8 = c.w_dtype == "fp8_e4m3_b128"
        for r in range(c.R):
            for l in range(c.L):
                for kind, tid, sid in weight_tensors(c):
                    np_view(image, self.view_fn(self.mode, r, l, tid))[...] = self.weight_view(r, l, kind)
                    if fp8:
                        np_view(image, self.view_fn(self.mode, r, l, sid))[...] = self.scale_view(r, l, kind)
                for m in self.attn_modes():
                    for kind, tid in ATTN_IDS.items():
                        np_view(image, self.view_fn(m, r, l, tid))[...] = self.attn_view(r, l, kind, m)
                for kvi in range(2):
                    pool, mask = self.pool(r, l, kvi)
                    np_view(image, self.view_fn(self.mode, r, l, 3 + kvi))[mask] = pool[mask]

    def compare(self, image: np.ndarray):
        """Bytewise comparison of every view of this mode; returns a list of mismatch strings.
        KV bytes outside the validity mask are unspecified (reading A10) and not compared."""
        c = self.st.cfg
        fp8 = c.w_dtype == "fp8_e4m3_b128"
        bad = []
        for r in range(c.R):
            for l in range(c.L):
                for kind, tid, sid in weight_tensors(c):
                    got = np_view(image, self.view_fn(self.mode, r, l, tid))
                    want = self.weight_view(r, l, kind)
                    if not np.array_equal(got.view(np.uint8), want.view(np.uint8)):
                        bad.append("weight r%d l%d %s: %d elems differ" % (r, l, kind, int((got != want).sum())))
                    if fp8:
                        got = np_view(image, self.view_fn(self.mode, r, l, sid))
                        want = self.scale_view(r, l, kind)
                        if not np.array_equal(got.view(np.uint32), want.view(np.uint32)):
                            bad.append("scale r%d l%d %s" % (r, l, kind))
                for m in self.attn_modes():
                    for kind, tid in ATTN_IDS.items():
                        got = np_view(image, self.view_fn(m, r, l, tid))
                        want = self.attn_view(r, l, kind, m)
                        if got.shape != want.shape or not np.array_equal(got, want):
                            bad.append("attn r%d l%d %s (%s view)" % (r, l, kind, "TP" if m == TP else "EP"))
                for kvi in range(2):
                    pool, mask = self.pool(r, l, kvi)
                    got = np_view(image, self.view_fn(self.mode, r, l, 3 + kvi))
                    if not np.array_equal(got[mask], pool[mask]):
                        bad.append("kv r%d l%d kv%d: %d slots differ" % (
                            r, l, kvi, int((got[mask] != pool[mask]).any(axis=(1, 2)).sum())))
        return bad


def target_request_state(st: State, to_mode: int, pages_tp: int, pages_ep: int, max_pages: int):
    """Oracle request state after a switch: owner and canonical tables (reading A7)."""
    c = st.cfg
    owner = okv.partition_requests(st.lens, c.R) if to_mode == EP else None
    bt = okv.canonical_block_tables(st.lens, owner, "ep" if to_mode == EP else "tp",
                                    pages_ep if to_mode == EP else pages_tp, c.page, max_pages)
    return owner, bt
