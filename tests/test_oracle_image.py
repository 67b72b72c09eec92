"""Negative controls for oracle/image.py (no GPU): `OracleLayout.compare` is what turns every parity
test red or green, so it must itself be seen red.  One flipped bit in each tensor kind (expert
weight, fp8 block scale, K/V pool inside the validity mask) is reported; an image that still holds
the SOURCE layout (a switch that did not happen) is reported; a flipped byte OUTSIDE the KV mask --
unspecified bytes, reading A10 -- and in spare / free space is not."""
import numpy as np
import pytest

import oracle
import workloads as wl
from harness import EP, TP, OracleLayout, State, mb, mb_config, source_tables


def layouts(cfg, fill="tag"):
    st = State(cfg, fill=fill)
    sess = mb.Session(mb_config(cfg, st.lens))      # host only: the library just reports the view offsets
    out = {}
    for mode in (TP, EP):
        owner, bt = source_tables(st, sess, mode, "random", seed=3)
        out[mode] = (OracleLayout(st, sess, mode, owner, bt), owner, bt)
    return st, sess, out


def flip(image, off, bit=0):
    image[off] ^= np.uint8(1 << bit)


@pytest.mark.parametrize("name,fill", [("tiny", "tag"), ("fp8", "normal"), ("w13", "tag")])
@pytest.mark.parametrize("mode", [TP, EP])
def test_compare_reports_single_bit_flips(name, fill, mode):
    cfg = {"tiny": wl.get_config("tiny"),
           "fp8": wl.get_config("fp8_graph").with_(L=1, E=8, H=128, I=1536, n_req=5, len_dist=("uniform", 1, 50), seed=4),
           "w13": wl.get_config("tiny").with_(w_orient=1, seed=6)}[name]
    st, sess, lay = layouts(cfg, fill)
    L, owner, bt = lay[mode]
    image = np.full(sess.layout.base_bytes, 0xA5, np.uint8)
    L.place(image)
    assert L.compare(image) == []
    c = st.cfg
    rng = np.random.default_rng(11)
    tensors = oracle.image.weight_tensors(c)
    kinds = [(tid, "weight") for _, tid, _ in tensors]
    if c.w_dtype == "fp8_e4m3_b128":
        kinds += [(sid, "scale") for _, _, sid in tensors]
    for tid, what in kinds:
        for r in range(c.R):
            v = sess.view_desc(mode, r, 0, tid)
            n = int(np.prod([v.shape[i] for i in range(v.ndim)])) * v.elem_bytes
            off = v.offset + int(rng.integers(n))
            bit = int(rng.integers(8))
            flip(image, off, bit)
            bad = L.compare(image)
            assert len(bad) == 1 and bad[0].startswith(what + " r%d l0" % r), (tid, r, bad)
            flip(image, off, bit)
    assert L.compare(image) == []
    # K / V pools: a flipped bit in a live slot is reported, one in a dead slot or a free page is not
    for kvi in range(2):
        for r in range(c.R):
            pool, mask = L.pool(r, 0, kvi)
            v = sess.view_desc(mode, r, 0, 3 + kvi)
            slot_bytes = int(np.prod(pool.shape[2:])) * v.elem_bytes
            live = np.argwhere(mask)
            dead = np.argwhere(~mask)
            if len(live):
                p, s = live[int(rng.integers(len(live)))]
                off = v.offset + (int(p) * c.page + int(s)) * slot_bytes + int(rng.integers(slot_bytes))
                flip(image, off, 5)
                bad = L.compare(image)
                assert len(bad) == 1 and bad[0].startswith("kv r%d l0 kv%d: 1 slots" % (r, kvi)), bad
                flip(image, off, 5)
            if len(dead):
                p, s = dead[int(rng.integers(len(dead)))]
                off = v.offset + (int(p) * c.page + int(s)) * slot_bytes + int(rng.integers(slot_bytes))
                flip(image, off, 5)
                assert L.compare(image) == []       # unspecified bytes (reading A10)
                flip(image, off, 5)
    sess.close()


@pytest.mark.parametrize("name", ["tiny", "w13"])
def test_compare_reports_an_image_that_was_not_switched(name):
    """The source layout left in place must not pass as the target layout: every weight view of every
    rank and every pool that holds a live token is reported."""
    cfg = wl.get_config("tiny") if name == "tiny" else wl.get_config("tiny").with_(w_orient=1, seed=6)
    st, sess, lay = layouts(cfg)
    c = st.cfg
    for src, dst in ((TP, EP), (EP, TP)):
        image = np.full(sess.layout.base_bytes, 0xA5, np.uint8)
        lay[src][0].place(image)
        bad = lay[dst][0].compare(image)
        n_w = sum(1 for b in bad if b.startswith("weight"))
        n_kv = sum(1 for b in bad if b.startswith("kv"))
        assert n_w == c.R * c.L * len(c.w_kinds), bad
        live_pools = sum(1 for r in range(c.R) for kvi in range(2) if lay[dst][0].pool(r, 0, kvi)[1].any())
        assert n_kv == live_pools and live_pools > 0, bad
    sess.close()


def test_compare_ignores_spare_slot_and_guard_bytes():
    """Bytes that belong to no view of the compared mode (the spare weight slot, the gap between the
    scale regions and the pools) are unspecified: changing them changes nothing."""
    st, sess, lay = layouts(wl.get_config("tiny"))
    L = lay[EP][0]
    image = np.full(sess.layout.base_bytes, 0xA5, np.uint8)
    L.place(image)
    covered = np.zeros(image.size, bool)
    c = st.cfg
    for r in range(c.R):
        for tid in (0, 1, 2, 3, 4):
            v = sess.view_desc(EP, r, 0, tid)
            n = int(np.prod([v.shape[i] for i in range(v.ndim)])) * v.elem_bytes
            covered[v.offset:v.offset + n] = True
    free = np.flatnonzero(~covered)
    assert free.size > 0
    image[free] ^= 0xFF
    assert L.compare(image) == []
    sess.close()
