"""Pins for oracle/attention.py (no GPU): a hand-worked fixture, the two figures the paper prints for
Qwen3-235B, brute-force index formulas, the head shards tiling the full tensor, and the
equivalence the layouts exist for -- tensor-parallel attention summed over ranks == data-parallel
attention == the dense block, in fp32 within 1e-5 -- with negative controls."""
import json
import os

import numpy as np
import pytest

import oracle
from oracle.attention import attn_forward_dense, attn_forward_ep, attn_forward_tp


def logical(Hq, Hkv, D, H, seed=0, dtype=np.float64):
    rng = np.random.default_rng(seed)
    return {k: rng.standard_normal(oracle.attn_shape(k, Hq, Hkv, D, H)).astype(dtype) * 0.3 for k in oracle.ATTN_KINDS}


def tp_views(W, R, Hq, Hkv):
    return [{k: oracle.attn_tp_view(W[k], k, r, R, Hq, Hkv) for k in oracle.ATTN_KINDS} for r in range(R)]


def test_golden_attention(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "attention_R2_Hq4_Hkv2_D2_H2.json")))
    R, Hq, Hkv, D, H = (g["inputs"][k] for k in ("R", "Hq", "Hkv", "D", "H"))
    W = {k: np.arange(int(np.prod(oracle.attn_shape(k, Hq, Hkv, D, H)))).reshape(oracle.attn_shape(k, Hq, Hkv, D, H))
         for k in oracle.ATTN_KINDS}
    e = g["expected"]
    for r in range(R):
        assert oracle.attn_tp_view(W["wq"], "wq", r, R, Hq, Hkv).ravel().tolist() == e["wq_tp"][r]
        assert oracle.attn_tp_view(W["wk"], "wk", r, R, Hq, Hkv).ravel().tolist() == e["wk_tp"][r]
        assert oracle.attn_tp_view(W["wk"], "wv", r, R, Hq, Hkv).ravel().tolist() == e["wk_tp"][r]
        assert oracle.attn_tp_view(W["wo"], "wo", r, R, Hq, Hkv).ravel().tolist() == e["wo_tp"][r]
        assert list(oracle.attn_tp_view(W["wq"], "wq", r, R, Hq, Hkv).shape) == e["wq_tp_shape"]
        assert list(oracle.attn_tp_view(W["wk"], "wk", r, R, Hq, Hkv).shape) == e["wk_tp_shape"]
        assert list(oracle.attn_tp_view(W["wo"], "wo", r, R, Hq, Hkv).shape) == e["wo_tp_shape"]
        for k in oracle.ATTN_KINDS:
            assert np.array_equal(oracle.attn_ep_view(W[k], r, R), W[k])


def test_paper_printed_sizes(golden_dir):
    """the q/k/v/o projections of Qwen3-235B total 'roughly 13 GB' in BF16 over 94 layers,
    and the TP shards held beside the full EP copies are '1.7 GB' per GPU (the paper truncates)."""
    g = json.load(open(os.path.join(golden_dir, "attention_R2_Hq4_Hkv2_D2_H2.json")))["paper_numbers"]
    a = oracle.attn_bytes(8, 94, 64, 4, 128, 4096, 2, "tp2ep", "dual")
    assert round(a["full_per_rank"] / 1e9) == g["full_GB_roughly"]
    assert int(a["duplicated_per_rank"] / 1e8) / 10 == g["tp_shard_GB"]
    assert a["moved"] == 0 and a["relocated"] == 0                     # pointer swap: nothing moves
    # "TP holds one-eighth per GPU" of q and o; the 4 KV heads on 8 ranks leave one head (a quarter) per rank
    q_or_o, k_or_v = 64 * 128 * 4096 * 2, 4 * 128 * 4096 * 2
    assert a["shard_per_rank"] == 94 * (2 * q_or_o // 8 + 2 * k_or_v // 4)


@pytest.mark.parametrize("R,Hq,Hkv", [(2, 4, 2), (4, 8, 2), (8, 16, 4), (4, 8, 8), (1, 4, 2), (4, 4, 1)])
def test_bruteforce_and_tiling(R, Hq, Hkv):
    D, H = 3, 5
    W = {k: np.arange(int(np.prod(oracle.attn_shape(k, Hq, Hkv, D, H))), dtype=np.int64).reshape(oracle.attn_shape(k, Hq, Hkv, D, H)) + 1000 * i
         for i, k in enumerate(oracle.ATTN_KINDS)}
    wq_rows, wo_cols, kv_seen = [], [], {}
    for r in range(R):
        vq, vk, vv, vo = (oracle.attn_tp_view(W[k], k, r, R, Hq, Hkv) for k in oracle.ATTN_KINDS)
        nq = Hq // R
        assert vq.shape == (nq, D, H) and vo.shape == (H, nq, D) and vq.flags["C_CONTIGUOUS"] and vo.flags["C_CONTIGUOUS"]
        for i in range(nq):                # per-element form: wq_tp[r][i][d][c] = wq[r*Hq/R + i][d][c]
            for d in range(D):
                for c in range(H):
                    assert vq[i, d, c] == W["wq"][r * nq + i, d, c]
                    assert vo[c, i, d] == W["wo"][c, r * nq + i, d]
        heads = [r * (Hkv // R) + i for i in range(Hkv // R)] if Hkv >= R else [r // (R // Hkv)]
        assert vk.shape == (len(heads), D, H)
        for i, h in enumerate(heads):
            assert np.array_equal(vk[i], W["wk"][h]) and np.array_equal(vv[i], W["wv"][h])
            kv_seen.setdefault(h, []).append(r)
        wq_rows.append(vq)
        wo_cols.append(vo)
    # the query-head shards tile wq and wo exactly; every KV head is held by R/Hkv ranks (or one)
    assert np.array_equal(np.concatenate(wq_rows, axis=0), W["wq"])
    assert np.array_equal(np.concatenate(wo_cols, axis=1), W["wo"])
    assert sorted(kv_seen) == list(range(Hkv)) and all(len(v) == max(1, R // Hkv) for v in kv_seen.values())


@pytest.mark.parametrize("R,Hq,Hkv", [(2, 4, 2), (4, 8, 2), (8, 16, 4), (4, 8, 8), (4, 4, 1)])
def test_tp_attention_equals_ep_equals_dense(R, Hq, Hkv):
    """PAPER.md:112 + :46: the TP layout (sum of rank partials over head shards) and the EP layout (the
    full copy on one rank) compute the same attention block: fp32 within 1e-5 relative of fp64 dense."""
    D, H, T = 8, 24, 6
    W64 = logical(Hq, Hkv, D, H, seed=R * 100 + Hq)
    x64 = np.random.default_rng(5).standard_normal((T, H))
    ref = attn_forward_dense(x64, *(W64[k] for k in oracle.ATTN_KINDS))
    W = {k: v.astype(np.float32) for k, v in W64.items()}
    x = x64.astype(np.float32)
    y_tp = attn_forward_tp(x, tp_views(W, R, Hq, Hkv), R, Hq, Hkv)
    y_ep = attn_forward_ep(x, {k: oracle.attn_ep_view(W[k], 0, R) for k in oracle.ATTN_KINDS})
    scale = np.abs(ref).max()
    assert np.abs(y_tp - ref).max() / scale <= 1e-5
    assert np.abs(y_ep - ref).max() / scale <= 1e-5


def test_negative_controls():
    """A plausible mistake in the layout breaks the equivalence: wo sharded along the wrong axis, query
    heads dealt round-robin instead of in blocks while wo stays blocked, the KV head of rank r taken as
    r mod Hkv instead of r div (R/Hkv)."""
    R, Hq, Hkv, D, H, T = 4, 8, 2, 8, 8, 5
    W = logical(Hq, Hkv, D, H, seed=9)
    x = np.random.default_rng(6).standard_normal((T, H))
    ref = attn_forward_dense(x, *(W[k] for k in oracle.ATTN_KINDS))
    good = tp_views(W, R, Hq, Hkv)
    assert np.abs(attn_forward_tp(x, good, R, Hq, Hkv) - ref).max() <= 1e-9
    nq = Hq // R
    bad = [dict(v) for v in good]
    for r in range(R):                       # (a) wo sliced along its OUTPUT axis H instead of the head axis
        bad[r]["wo"] = np.ascontiguousarray(W["wo"][r * (H // R):(r + 1) * (H // R)].reshape(-1)[:H * nq * D].reshape(H, nq, D))
    assert np.abs(attn_forward_tp(x, bad, R, Hq, Hkv) - ref).max() > 1e-3
    bad = [dict(v) for v in good]
    for r in range(R):                       # (b) round-robin query heads
        bad[r]["wq"] = np.ascontiguousarray(W["wq"][r::R])
    assert np.abs(attn_forward_tp(x, bad, R, Hq, Hkv) - ref).max() > 1e-3
    bad = [dict(v) for v in good]
    for r in range(R):                       # (c) KV head r mod Hkv
        bad[r]["wk"] = np.ascontiguousarray(W["wk"][[r % Hkv]])
        bad[r]["wv"] = np.ascontiguousarray(W["wv"][[r % Hkv]])
    assert np.abs(attn_forward_tp(x, bad, R, Hq, Hkv) - ref).max() > 1e-3


def test_gather_variant_bytes_closed_form():
    """Memory-saving variant (PAPER.md:112 'rebuilds TP-EP with an All-Gather'): every rank receives the
    heads it does not hold: (Hq - Hq/R) heads of wq and of wo, (Hkv - held) heads of wk and of wv; nothing
    moves EP->TP (the local slice stays in place, reading A19)."""
    for (R, L, Hq, Hkv, D, H, b) in [(8, 3, 64, 4, 128, 4096, 2), (4, 2, 8, 8, 16, 32, 2), (2, 1, 4, 2, 2, 2, 4), (1, 1, 4, 2, 2, 2, 2)]:
        head = D * H * b
        held_kv = Hkv // R if Hkv >= R else 1
        want = L * R * (2 * (Hq - Hq // R) + 2 * (Hkv - held_kv)) * head
        a = oracle.attn_bytes(R, L, Hq, Hkv, D, H, b, "tp2ep", "gather")
        assert a["moved"] == a["relocated"] == a["read"] == want
        z = oracle.attn_bytes(R, L, Hq, Hkv, D, H, b, "ep2tp", "gather")
        assert z["moved"] == z["relocated"] == 0 and z["duplicated_per_rank"] == 0
