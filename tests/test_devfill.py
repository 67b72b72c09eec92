"""The test-only device fill (tests/devfill.py) against the oracle, on CPU tensors: what it writes
into the TP views of a buffer is exactly the TP layout the oracle builds from the tag-filled logical
tensors.  (The full-size GPU tests rely on it for their source state.)"""
import numpy as np
import pytest

import devfill
import workloads as wl
from harness import TP, OracleLayout, State, mb, mb_config

torch = pytest.importorskip("torch")


@pytest.mark.parametrize("name,kw", [
    ("tiny", {}),
    ("small", dict(L=2, H=64, I=128, n_req=9, len_dist=("uniform", 1, 90))),
    ("fp8_graph", dict(L=1, E=8, H=128, I=1536, n_req=7, len_dist=("uniform", 1, 70))),
    ("small", dict(L=2, H=64, I=128, n_req=9, len_dist=("uniform", 1, 90), w_orient=1)),
])
def test_devfill_equals_oracle_tp_layout(name, kw):
    cfg = wl.get_config(name).with_(**kw)
    st = State(cfg, fill="tag")
    sess = mb.Session(mb_config(cfg, st.lens))
    sess.base = torch.zeros(sess.layout.base_bytes, dtype=torch.uint8)      # a CPU stand-in for the device buffer
    devfill.fill_random(sess)
    mp = sess.cfg.max_pages_per_request
    bt = wl.random_page_tables(st.lens, None, cfg.R, sess.layout.pages_tp, cfg.page, mp, seed=5)
    for l in range(cfg.L):
        for kind in cfg.w_kinds:
            devfill.fill_tp_weight(sess, cfg, l, kind, experts_per_chunk=3)
        for kvi in range(2):
            devfill.fill_tp_pool(sess, cfg, l, kvi, st.lens, bt, tokens_per_chunk=50)
    image = sess.base.numpy()
    lay = OracleLayout(st, sess, TP, None, bt)
    if cfg.w_dtype == "fp8_e4m3_b128":      # scales are not tag-filled: take the oracle's
        for r in range(cfg.R):
            for l in range(cfg.L):
                for m, kind in enumerate(devfill.KINDS):
                    v = sess.view_desc(TP, r, l, 5 + m)
                    n = int(np.prod([v.shape[i] for i in range(v.ndim)])) * 4
                    image[v.offset:v.offset + n] = np.ascontiguousarray(lay.scale_view(r, l, kind)).view(np.uint8).reshape(-1)
    bad = lay.compare(image)
    assert not bad, bad[:5]
    t0 = devfill.TENSOR_ID[cfg.w_kinds[0]]
    a = devfill.weighted_checksum(sess.view(TP, 0, 0, t0))
    v = sess.view(TP, 0, 0, t0)
    v[0, 0, 0], v[0, 0, 1] = v[0, 0, 1].clone(), v[0, 0, 0].clone()
    b = devfill.weighted_checksum(v)
    assert a[0] == b[0] and (a[1] != b[1] or int(v[0, 0, 0]) == int(v[0, 0, 1]))
    sess.close()
