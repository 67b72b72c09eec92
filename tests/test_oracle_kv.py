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


def test_scale_bytes_closed_forms():
    """oracle.scale_bytes (SURVEY.md §8(c) "(+ scales)", reading A13) against closed forms worked by hand.

    I/R = 192 (I = 1536, R = 8; the Qwen3-235B shape): shard j covers columns [192j, 192j+191], i.e.
    blocks {0,1} {1,2} {3,4} {4,5} {6,7} {7,8} {9,10} {10,11}: 2 blocks per shard, 16 holder slots for
    the 12 blocks; blocks 1, 4, 7, 10 are straddled.  Lowest holders of blocks 0..11:
    0 0 1 2 2 3 4 4 5 6 6 7 -- every block has ONE source rank, which owns E/R of the experts itself.
      ep2tp: relocated = 16 slots, moved = 16 * (1 - 1/R), read = 12 (each source block once)
      tp2ep: relocated = read = 12, moved = 12 * (1 - 1/R)          [per expert, x H/128 * 4 bytes]
    Aligned shape (I/R a multiple of 128): no block is shared, both directions move (1 - 1/R) of
    E * I/128 * H/128 * 4 bytes, exactly like the weights."""
    R, L, E, H, I = 8, 4, 128, 4096, 1536
    blk = (H // 128) * 4
    for kinds, f in ((("gate", "up", "down"), 3), (("w13", "w2"), 3), (("down",), 1)):
        e2t = oracle.scale_bytes(R, L, E, H, I, "ep2tp", kinds)
        t2e = oracle.scale_bytes(R, L, E, H, I, "tp2ep", kinds)
        assert e2t == {"relocated": L * f * E * 16 * blk, "moved": L * f * (E - E // R) * 16 * blk,
                       "read": L * f * E * 12 * blk}
        assert t2e == {"relocated": L * f * E * 12 * blk, "moved": L * f * (E - E // R) * 12 * blk,
                       "read": L * f * E * 12 * blk}
    # BASELINE.json config 5: 2.36 MB of scales in total
    assert oracle.scale_bytes(8, 4, 128, 4096, 1536, "tp2ep")["relocated"] == 2359296
    for (R, L, E, H, I) in [(4, 2, 8, 256, 1024), (2, 1, 4, 128, 256), (8, 1, 8, 128, 1024)]:
        assert (I // R) % 128 == 0
        tot = L * 3 * E * (I // 128) * (H // 128) * 4
        for d in ("ep2tp", "tp2ep"):
            a = oracle.scale_bytes(R, L, E, H, I, d)
            assert a["relocated"] == tot and a["read"] == tot and a["moved"] * R == tot * (R - 1)
    # R = 1: one rank holds everything, nothing changes owner
    a = oracle.scale_bytes(1, 1, 4, 128, 256, "ep2tp")
    assert a["moved"] == 0 and a["relocated"] == 3 * 4 * 2 * 1 * 4


@pytest.mark.parametrize("R,E,H,I", [(8, 16, 256, 1536), (4, 8, 128, 768), (8, 8, 128, 2048), (2, 4, 256, 384)])
def test_scale_bytes_equal_the_scale_views(R, E, H, I):
    """Reduction onto the separately pinned views (tp_scale_view is pinned by the dequantised-shard
    equality in test_oracle_weights.py): EP->TP writes exactly the TP scale views, TP->EP exactly the
    EP scale views; and the owner-changed part counted by brute force over explicit owner arrays."""
    L = 1
    for kinds in (("gate", "up", "down"), ("w13", "w2")):
        tp_bytes = ep_bytes = moved_e2t = moved_t2e = 0
        for kind in kinds:
            mult = 2 if kind == "w13" else 1
            shape = (E, H // 128, I // 128) if kind in ("gate", "up", "w2") else (E, mult * I // 128, H // 128)
            S = np.arange(int(np.prod(shape)), dtype=np.float32).reshape(shape)
            ids = np.arange(S.size).reshape(shape).astype(np.float32)        # identity of every scale
            owner_of = np.repeat(np.arange(R), E // R)                       # EP owner of expert e
            first_holder = {}
            for j in range(R):
                v = oracle.tp_scale_view(ids, kind, j, R, I)
                tp_bytes += v.nbytes
                q = np.broadcast_to(owner_of.reshape(-1, 1, 1), v.shape)
                moved_e2t += int((q != j).sum()) * 4
                for x, qq in zip(v.ravel().tolist(), q.ravel().tolist()):
                    first_holder.setdefault(x, (j, qq))                      # lowest rank seen first
                ep_bytes += oracle.ep_scale_view(S, j, R).nbytes
            assert len(first_holder) == S.size
            moved_t2e += sum(4 for (j, qq) in first_holder.values() if j != qq)
        e2t = oracle.scale_bytes(R, L, E, H, I, "ep2tp", kinds)
        t2e = oracle.scale_bytes(R, L, E, H, I, "tp2ep", kinds)
        assert (e2t["relocated"], e2t["moved"], e2t["read"]) == (tp_bytes, moved_e2t, ep_bytes)
        assert (t2e["relocated"], t2e["moved"], t2e["read"]) == (ep_bytes, moved_t2e, ep_bytes)
