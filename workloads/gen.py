"""Seeded random draws.  No layout / partition / allocation arithmetic lives here."""
from __future__ import annotations

import numpy as np

from .configs import Config


def bf16_bits_from_f32(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16, returned as uint16 bit patterns (numpy has no bf16)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    rounded = u + (np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1)))
    return (rounded >> np.uint32(16)).astype(np.uint16)


def _np_dtype(w_dtype: str):
    return {"bf16": np.uint16, "fp32": np.float32, "fp8_e4m3_b128": np.uint8}[w_dtype]


def tag_fill_u16(shape, salt: int) -> np.ndarray:
    """Coordinate-tag fill: element value = 16-bit hash of (salt, flat logical index).

    Random bf16 values repeat; a tag makes a misplaced element visible.
    Generated in blocks so that a full-size tensor (8e8 elements) needs no multi-GB temporaries."""
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.uint16)
    off = np.uint64((int(salt) * 0x9E3779B97F4A7C15) & 0xFFFFFFFFFFFFFFFF)
    step = 1 << 24
    with np.errstate(over="ignore"):
        for a in range(0, n, step):
            h = np.arange(a, min(n, a + step), dtype=np.uint64) + off
            h ^= h >> np.uint64(33)
            h *= np.uint64(0xFF51AFD7ED558CCD)
            h ^= h >> np.uint64(29)
            out[a:a + step] = (h & np.uint64(0xFFFF)).astype(np.uint16)
    return out.reshape(shape)


def tag_salt_offset(salt: int) -> int:
    """The additive offset tag_fill_u16 derives from a salt, as a signed 64-bit integer."""
    off = (int(salt) * 0x9E3779B97F4A7C15) & 0xFFFFFFFFFFFFFFFF
    return off - (1 << 64) if off >= (1 << 63) else off


def tag_fill_u16_torch(flat_index, offset):
    """The same counter-based generator as tag_fill_u16, on torch int64 tensors (any device):
    `flat_index` = flat logical index of each element, `offset` = tag_salt_offset(salt) (a Python
    int or a broadcastable int64 tensor).  Returns int64 values in [0, 65535].  int64 arithmetic
    wraps like uint64; logical right shifts are arithmetic shifts with the sign bits masked off."""
    h = flat_index + offset
    h = h ^ ((h >> 33) & 0x7FFFFFFF)
    h = h * (0xFF51AFD7ED558CCD - (1 << 64))
    h = h ^ ((h >> 29) & ((1 << 35) - 1))
    return h & 0xFFFF


_KIND_ID = {"gate": 0, "up": 1, "down": 2, "w13": 3, "w2": 4}


def weight_shape(cfg: Config, kind: str) -> tuple:
    """Logical shape of one layer's expert tensor: gate/up [E,H,I], down [E,I,H] (BASELINE.json);
    w13 [E,2I,H], w2 [E,H,I] (the paper's own orientation)."""
    return {"gate": (cfg.E, cfg.H, cfg.I), "up": (cfg.E, cfg.H, cfg.I), "down": (cfg.E, cfg.I, cfg.H),
            "w13": (cfg.E, 2 * cfg.I, cfg.H), "w2": (cfg.E, cfg.H, cfg.I)}[kind]


def weight_tag_salt(cfg: Config, layer: int, kind: str) -> int:
    m = _KIND_ID[kind]
    if m < 3:
        return cfg.seed * 1000 + layer * 3 + m
    return cfg.seed * 1000 + 500 + layer * 2 + (m - 3)


def kv_tag_salt(cfg: Config, layer: int, kv: int, req: int) -> int:
    return cfg.seed * 7919 + (layer * 2 + kv) * 100003 + req


def gen_logical_weight(cfg: Config, layer: int, kind: str, fill: str = "normal") -> np.ndarray:
    """Logical expert tensor of one layer: gate/up [E,H,I], down [E,I,H] (BASELINE.json orientation).

    bf16 -> uint16 bit patterns of N(0, 0.02); fp32 -> float32 N(0, 0.02); fp8 -> uint8 bytes
    (opaque e4m3 codes, uniform over 0..255 minus the two NaN codes)."""
    m = _KIND_ID[kind]
    shape = weight_shape(cfg, kind)
    seed = (cfg.seed, 2000 + layer, m)
    if fill == "tag":
        t = tag_fill_u16(shape, salt=weight_tag_salt(cfg, layer, kind))
        if cfg.w_dtype == "bf16":
            return t
        if cfg.w_dtype == "fp8_e4m3_b128":
            return (t & 0xFF).astype(np.uint8)
        return t.astype(np.float32)
    rng = np.random.default_rng(seed)
    if cfg.w_dtype == "fp8_e4m3_b128":
        b = rng.integers(0, 256, size=shape, dtype=np.uint8)
        b[(b & 0x7F) == 0x7F] = 0x38  # avoid NaN codes; bytes are opaque to the reshard anyway
        return b
    x = rng.normal(0.0, 0.02, size=shape).astype(np.float32)
    return x if cfg.w_dtype == "fp32" else bf16_bits_from_f32(x)


def gen_logical_scale(cfg: Config, layer: int, kind: str) -> np.ndarray:
    """fp32 per-128x128-block scales: gate/up [E, H/128, I/128], down [E, I/128, H/128];
    w13 [E, 2I/128, H/128], w2 [E, H/128, I/128]."""
    m = _KIND_ID[kind]
    shape = tuple([cfg.E] + [d // 128 for d in weight_shape(cfg, kind)[1:]])
    rng = np.random.default_rng((cfg.seed, 2500 + layer, m))
    return rng.uniform(0.5, 2.0, size=shape).astype(np.float32)


_ATTN_ID = {"wq": 0, "wk": 1, "wv": 2, "wo": 3}


def attn_weight_shape(cfg: Config, kind: str) -> tuple:
    """Logical attention projections of one layer: wq [Hq,D,H], wk/wv [Hkv,D,H], wo [H,Hq,D]."""
    Hq, Hkv, D, H = cfg.n_q_heads, cfg.kv_heads, cfg.head_dim, cfg.H
    return {"wq": (Hq, D, H), "wk": (Hkv, D, H), "wv": (Hkv, D, H), "wo": (H, Hq, D)}[kind]


def attn_tag_salt(cfg: Config, layer: int, kind: str) -> int:
    return cfg.seed * 1000 + 700 + layer * 4 + _ATTN_ID[kind]


def gen_attn_weight(cfg: Config, layer: int, kind: str, fill: str = "tag") -> np.ndarray:
    """bf16 bit patterns (uint16) of one attention projection: coordinate tags, or N(0, 0.02)."""
    shape = attn_weight_shape(cfg, kind)
    if fill == "tag":
        return tag_fill_u16(shape, salt=attn_tag_salt(cfg, layer, kind))
    rng = np.random.default_rng((cfg.seed, 2700 + layer, _ATTN_ID[kind]))
    return bf16_bits_from_f32(rng.normal(0.0, 0.02, size=shape).astype(np.float32))


def draw_seq_lens(cfg: Config, n_req: int | None = None) -> np.ndarray:
    """Request lengths in tokens (int32), numpy.random.default_rng(cfg.seed)."""
    n = cfg.n_req if n_req is None else n_req
    rng = np.random.default_rng(cfg.seed)
    d = cfg.len_dist
    if d[0] == "uniform":
        x = rng.integers(d[1], d[2] + 1, size=n)
    elif d[0] == "lognormal":
        x = np.rint(rng.lognormal(np.log(d[1]), d[2], size=n))
        x = np.clip(x, 1, d[3])
    elif d[0] == "geometric":
        x = np.clip(rng.geometric(1.0 / d[1], size=n), 1, d[2])
    else:
        raise ValueError(d)
    return x.astype(np.int32)


def gen_kv_request(cfg: Config, layer: int, kv: int, req: int, length: int,
                   fill: str = "normal") -> np.ndarray:
    """K (kv=0) or V (kv=1) of one request in one layer: [len, kv_heads, head_dim] bf16 bits."""
    shape = (int(length), cfg.kv_heads, cfg.head_dim)
    if fill == "tag":
        return tag_fill_u16(shape, salt=kv_tag_salt(cfg, layer, kv, req))
    rng = np.random.default_rng((cfg.seed, 3000 + layer, kv, req))
    return bf16_bits_from_f32(rng.normal(0.0, 1.0, size=shape).astype(np.float32))


def random_page_tables(seq_lens, owner, n_ranks: int, n_pages: int, page: int, max_pages: int,
                       seed: int) -> np.ndarray:
    """Seeded random injective page assignment (reading A8: pages 'interleave arbitrarily',
    PAPER.md:122).  `owner[i] < 0` means every rank uses the same table (one shared draw);
    otherwise pages are drawn per owning rank.  Returns int32 [n, max_pages], -1 padded."""
    rng = np.random.default_rng(seed)
    seq_lens = np.asarray(seq_lens)
    n = len(seq_lens)
    bt = np.full((n, max_pages), -1, dtype=np.int32)
    need = (seq_lens + page - 1) // page
    groups = {}
    for i in range(n):
        groups.setdefault(int(owner[i]) if owner is not None else -1, []).append(i)
    for g, members in sorted(groups.items()):
        total = int(sum(need[i] for i in members))
        if total > n_pages:
            raise ValueError("pool too small for the random source tables")
        perm = rng.permutation(n_pages)[:total]
        k = 0
        for i in members:
            bt[i, :need[i]] = perm[k:k + need[i]]
            k += need[i]
    return bt


def kv_pool_bytes(cfg: Config, seq_lens, policy: str | None = None) -> int:
    """Capacity of one K (or V) pool of one rank and layer (a workload parameter BASELINE.json
    leaves open).  "roomy": 1.1 x (TP need + an upper bound of the largest EP
    share), so source and target pages never have to overlap; "tight": 1.05 x TP need, which
    forces dependency rounds and staging.  Rounded up to whole EP pages."""
    policy = policy or cfg.pool_policy
    seq_lens = np.asarray(seq_lens, dtype=np.int64)
    b = cfg.kv_elem_bytes
    hpr = max(1, cfg.kv_heads // cfg.R)
    tp_page = cfg.page * hpr * cfg.head_dim * b
    ep_page = cfg.page * cfg.kv_heads * cfg.head_dim * b
    pages = (seq_lens + cfg.page - 1) // cfg.page
    total = int(pages.sum())
    biggest = int(pages.max()) if len(pages) else 0
    tp_need = total * tp_page
    ep_share = (-(-total // cfg.R) + biggest) * ep_page   # LPT bound on the fullest rank
    if policy == "roomy":
        need = 1.1 * (tp_need + ep_share)
    elif policy == "tight":
        need = max(1.05 * tp_need, ep_share)
    else:
        raise ValueError(policy)
    n_pages = max(1, int(-(-need // ep_page)))
    return n_pages * ep_page
