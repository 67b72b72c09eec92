"""Pins for oracle/kv.py and oracle/accounting.py (no GPU): hand-worked fixtures, reachability /
round-trip invariants, partition properties, closed forms."""
import json
import os

import numpy as np
import pytest

import oracle
import workloads as wl


def _g(golden_dir, name):
    return json.load(open(os.path.join(golden_dir, name)))


def test_golden_kv_heads(golden_dir):
    g = _g(golden_dir, "kv_heads.json")
    for c in g["cases"]:
        got = [oracle.kv_heads_of_rank(r, c["R"], c["Hkv"]) for r in range(c["R"])]
        assert got == c["heads"]
    s = g["tp_source_rank"]
    for c in s["cases"]:
        assert oracle.tp_source_rank(c["head"], c["owner"], s["R"], s["Hkv"]) == c["src"]


def test_golden_partition_and_tables(golden_dir):
    g = _g(golden_dir, "partition_and_tables.json")
    for c in g["partition"]:
        assert oracle.partition_requests(c["seq_lens"], c["R"]).tolist() == c["owner"]
    t = g["tables"]
    bt = oracle.canonical_block_tables(t["seq_lens"], None, "tp", t["tp"]["n_pages"], t["page"], t["max_pages"])
    assert bt.tolist() == t["tp"]["bt"]
    bt = oracle.canonical_block_tables(t["seq_lens"], t["ep"]["owner"], "ep", t["ep"]["n_pages"], t["page"],
                                       t["max_pages"])
    assert bt.tolist() == t["ep"]["bt"]
    # capacity: TP needs 10 pages, rank 1 under EP needs 5
    with pytest.raises(oracle.CapacityError):
        oracle.canonical_block_tables(t["seq_lens"], None, "tp", 9, t["page"], t["max_pages"])
    with pytest.raises(oracle.CapacityError):
        oracle.canonical_block_tables(t["seq_lens"], t["ep"]["owner"], "ep", 4, t["page"], t["max_pages"])


def test_golden_pool_images(golden_dir):
    g = _g(golden_dir, "kv_pool_images.json")
    i = g["inputs"]
    K = {0: np.array(i["K"]).reshape(i["len"], i["Hkv"], i["D"])}
    lens = [i["len"]]
    for r in range(i["R"]):
        pool, mask = oracle.tp_pool_image(K, lens, [g["tp"]["bt"]], r, i["R"], i["Hkv"], i["D"], i["page"],
                                          i["n_pages"])
        want = g["tp"]["rank%d" % r]
        m = np.array(want["mask"], bool)
        assert mask.ravel().tolist() == m.tolist()
        assert pool.reshape(-1)[np.repeat(m, 1)].tolist() == np.array(want["pool"])[m].tolist()
        pool, mask = oracle.ep_pool_image(K, lens, [g["ep"]["owner"]], [g["ep"]["bt"]], r, i["Hkv"], i["D"],
                                          i["page"], i["n_pages"])
        want = g["ep"]["rank%d" % r]
        m = np.array(want["mask"], bool)
        assert mask.ravel().tolist() == m.tolist()
        m2 = np.repeat(m, i["Hkv"] * i["D"])
        assert pool.reshape(-1)[m2].tolist() == np.array(want["pool"])[m2].tolist()


@pytest.mark.parametrize("name", ["tiny", "small"])
def test_partition_properties(name):
    cfg = wl.get_config(name)
    lens = wl.draw_seq_lens(cfg)
    R = cfg.R
    o1 = oracle.partition_requests(lens, R)
    o2 = oracle.partition_requests(lens.copy(), R)
    assert np.array_equal(o1, o2)                       # deterministic
    assert o1.min() >= 0 and o1.max() < R               # disjoint cover: one owner each
    tok = np.bincount(o1, weights=lens, minlength=R)
    assert tok.max() - tok.min() <= lens.max()          # LPT bound
    cnt = np.bincount(o1, minlength=R)
    assert cnt.max() - cnt.min() <= max(2, len(lens) // R)


def test_partition_tiny_hand_computed():
    """Expectation written from the generated lengths (SURVEY.md §8(c) 'partition' pin)."""
    cfg = wl.get_config("tiny")
    lens = wl.draw_seq_lens(cfg).tolist()
    # by hand: visit in (-len, id) order, keep (tokens, reqs) per rank
    order = sorted(range(4), key=lambda i: (-lens[i], i))
    load = [[0, 0], [0, 0]]
    want = [None] * 4
    for i in order:
        r = 0 if (load[0][0], load[0][1]) <= (load[1][0], load[1][1]) else 1
        want[i] = r
        load[r][0] += lens[i]
        load[r][1] += 1
    assert oracle.partition_requests(lens, 2).tolist() == want
    assert sorted(want) == [0, 0, 1, 1]


def _logical_kv(cfg, lens, layer=0, kv=0, fill="tag"):
    return {i: wl.gen_kv_request(cfg, layer, kv, i, int(lens[i]), fill=fill) for i in range(len(lens))}


@pytest.mark.parametrize("lens", [None, [1, 16, 17, 32, 33, 0]])
def test_reachability_and_round_trip_tiny(lens):
    """PAPER.md:126 'no request is dropped'; PAPER.md:96 KV values 'the same before and after'.
    Covers len = 1, k*pg, k*pg+1 and a waiting request (len 0)."""
    cfg = wl.get_config("tiny")
    R, Hkv, D, pg = cfg.R, cfg.kv_heads, cfg.head_dim, cfg.page
    lens = wl.draw_seq_lens(cfg) if lens is None else np.array(lens, dtype=np.int32)
    KV = _logical_kv(cfg, lens)
    max_pages = 8
    need = sum(oracle.pages_needed(x, pg) for x in lens)
    n_tp, n_ep = need + 3, need + 1
    owner = oracle.partition_requests(lens, R)
    bt_tp = oracle.canonical_block_tables(lens, None, "tp", n_tp, pg, max_pages)
    bt_ep = oracle.canonical_block_tables(lens, owner, "ep", n_ep, pg, max_pages)
    # tables: in range, injective per rank, -1 beyond the need
    for i, n in enumerate(lens):
        k = oracle.pages_needed(n, pg)
        assert np.all(bt_tp[i, k:] == -1) and np.all(bt_ep[i, k:] == -1)
        assert np.all((bt_tp[i, :k] >= 0) & (bt_tp[i, :k] < n_tp))
        assert np.all((bt_ep[i, :k] >= 0) & (bt_ep[i, :k] < n_ep))
    live = bt_tp[bt_tp >= 0]
    assert len(set(live.tolist())) == len(live)
    for r in range(R):
        live = bt_ep[owner == r]
        live = live[live >= 0]
        assert len(set(live.tolist())) == len(live)
    tp = [oracle.tp_pool_image(KV, lens, bt_tp, r, R, Hkv, D, pg, n_tp) for r in range(R)]
    ep = [oracle.ep_pool_image(KV, lens, owner, bt_ep, r, Hkv, D, pg, n_ep) for r in range(R)]
    # valid-slot counts: TP every rank holds every token; EP only the owner's
    for r in range(R):
        assert tp[r][1].sum() == lens.sum()
        assert ep[r][1].sum() == lens[owner == r].sum()
    # reachability: gather through the tables reproduces the logical KV from either layout
    for i, n in enumerate(lens):
        a = oracle.gather_request_from_tp([p for p, _ in tp], bt_tp[i], int(n), R, Hkv, D, pg)
        b = oracle.gather_request_from_ep(ep[owner[i]][0], bt_ep[i], int(n), pg)
        assert np.array_equal(a, KV[i]) and np.array_equal(b, KV[i])
    # TP->EP->TP: rebuilding TP from the KV gathered out of EP gives the identical TP image
    KV2 = {i: oracle.gather_request_from_ep(ep[owner[i]][0], bt_ep[i], int(lens[i]), pg) for i in range(len(lens))}
    for r in range(R):
        p2, m2 = oracle.tp_pool_image(KV2, lens, bt_tp, r, R, Hkv, D, pg, n_tp)
        assert np.array_equal(m2, tp[r][1]) and np.array_equal(p2, tp[r][0])


def test_replicated_heads_agree():
    cfg = wl.get_config("tiny").with_(R=4, kv_heads=2)  # 2 ranks per head
    lens = np.array([5, 20], dtype=np.int32)
    KV = _logical_kv(cfg, lens)
    bt = oracle.canonical_block_tables(lens, None, "tp", 4, cfg.page, 2)
    pools = [oracle.tp_pool_image(KV, lens, bt, r, 4, 2, cfg.head_dim, cfg.page, 4)[0] for r in range(4)]
    assert np.array_equal(pools[0], pools[1]) and np.array_equal(pools[2], pools[3])
    assert not np.array_equal(pools[0], pools[2])
    assert pools[0].shape == (4, 16, 1, 16)


def test_weight_bytes_closed_form():
    """(1 - 1/R) * L*3*E*H*I*b owner-changed; all bytes relocate."""
    for (R, L, E, H, I, b) in [(2, 1, 8, 64, 32, 2), (4, 4, 16, 64, 32, 2), (8, 2, 16, 8, 24, 1), (1, 1, 2, 4, 4, 2)]:
        tot = L * 3 * E * H * I * b
        for d in ("ep2tp", "tp2ep"):
            a = oracle.weight_bytes(R, L, E, H, I, b, d)
            assert a["relocated"] == tot and a["read"] == tot
            assert a["moved"] * R == tot * (R - 1)


def test_kv_bytes_closed_form():
    """per token per layer (K and V): Hkv<R: EP->TP (R-1)*2*D*b, TP->EP
    (Hkv-1)*2*D*b; Hkv>=R: Hkv*(1-1/R)*2*D*b both ways."""
    lens = np.array([3, 10, 7, 1, 16], dtype=np.int32)
    T = int(lens.sum())
    for (R, Hkv) in [(8, 4), (2, 2), (4, 8), (4, 1), (1, 2)]:
        owner = oracle.partition_requests(lens, R)
        D, b, L = 16, 2, 3
        e2t = oracle.kv_bytes(lens, owner, R, L, Hkv, D, b, "ep2tp")
        t2e = oracle.kv_bytes(lens, owner, R, L, Hkv, D, b, "tp2ep")
        if Hkv < R:
            assert e2t["moved"] == T * L * (R - 1) * 2 * D * b
            assert t2e["moved"] == T * L * (Hkv - 1) * 2 * D * b
            assert e2t["relocated"] == T * L * R * 2 * D * b
        else:
            assert e2t["moved"] * R == T * L * Hkv * (R - 1) * 2 * D * b
            assert t2e["moved"] == e2t["moved"]
            assert e2t["relocated"] == T * L * Hkv * 2 * D * b
        assert t2e["relocated"] == T * L * Hkv * 2 * D * b
        assert e2t["read"] == T * L * Hkv * 2 * D * b and t2e["read"] == T * L * Hkv * 2 * D * b
