"""The C-ABI boundary without a GPU: the library loads, exports every symbol include/moebius.h
declares (and nothing else under the moebius_ prefix is missing from the header), the host-only
entry points behave as the header says, and the product path has no route into oracle/."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

import workloads as wl
from harness import EP, TP, mb, mb_config

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "moebius.h")


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"MOEBIUS_API\s+[\w\s\*]+?\b(moebius_\w+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for must in ("moebius_plan", "moebius_reshard", "moebius_block_tables"):
        assert must in names
    assert len(names) >= 15


def test_library_exports_every_declared_symbol():
    so = C.CDLL(mb.lib_path())
    for name in declared_symbols():
        assert getattr(so, name) is not None, name
    assert sorted(mb.EXPORTED_SYMBOLS) == declared_symbols()


def test_no_undeclared_exports():
    out = subprocess.run(["nm", "-D", "--defined-only", mb.lib_path()], capture_output=True, text=True).stdout
    exported = sorted(l.split()[-1] for l in out.splitlines() if " T " in l and "moebius_" in l.split()[-1]
                      and not l.split()[-1].startswith("_Z"))
    assert exported == declared_symbols()


def test_header_is_plain_c():
    """extern "C", plain pointers and sizes, no torch / C++ types: the header compiles as C."""
    src = "#include \"%s\"\nint main(void){ moebius_config_t c; c.struct_size = sizeof c; return (int)c.struct_size == 0; }\n" % HEADER
    r = subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-fsyntax-only", "-x", "c", "-"], input=src,
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr


def test_struct_sizes_match_the_header():
    src = ("#include <stdio.h>\n#include \"%s\"\nint main(void){ printf(\"%%zu %%zu %%zu %%zu\\n\", sizeof(moebius_config_t),"
           " sizeof(moebius_layout_t), sizeof(moebius_view_t), sizeof(moebius_stats_t)); return 0; }\n" % HEADER)
    exe = os.path.join(ROOT, "tests", "emul", "abi_sizes.out")
    r = subprocess.run(["gcc", "-std=c99", "-x", "c", "-", "-o", exe], input=src, capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    sizes = [int(x) for x in subprocess.run([exe], capture_output=True, text=True).stdout.split()]
    os.remove(exe)
    assert sizes == [C.sizeof(mb.moebius_config_t), C.sizeof(mb.moebius_layout_t), C.sizeof(mb.moebius_view_t),
                     C.sizeof(mb.moebius_stats_t)]


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_26607_b200")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cpp", ".cu", ".h")):
                text = open(os.path.join(d, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "oracle/" not in text.replace("shares nothing with oracle/", "").replace(
                    "CPU oracle under oracle/", "").replace("imports `oracle/`", ""), f
    assert not re.search(r"^\s*(import|from)\s+oracle\b", open(os.path.join(ROOT, "workloads", "gen.py")).read(), flags=re.M)


def tiny_cfg(**kw):
    cfg = wl.get_config("tiny")
    lens = wl.draw_seq_lens(cfg)
    c = mb_config(cfg, lens)
    for k, v in kw.items():
        setattr(c, k, v)
    return cfg, lens, c


@pytest.mark.parametrize("field,value", [("R", 3), ("I", 24), ("w_orient", 2), ("kv_heads", 3), ("page_tokens", 0),
                                         ("page_tokens", 256), ("w_dtype", 9), ("kv_dtype", 2), ("R", 0),
                                         ("kv_pool_bytes_per_rank_layer", 1000)])
def test_create_rejects_bad_configs(field, value):
    """Reading A3: E % R, I % R, 16-byte runs, head geometry, pool a whole number of EP pages."""
    _, _, c = tiny_cfg(**{field: value})
    with pytest.raises(mb.MoebiusError) as e:
        mb.moebius_create(c)
    assert e.value.status == -1


def test_struct_size_is_checked():
    _, _, c = tiny_cfg()
    c.struct_size = 8
    out = C.c_void_p()
    so = C.CDLL(mb.lib_path())
    so.moebius_create.argtypes = [C.c_void_p, C.c_void_p]
    assert so.moebius_create(C.byref(c), C.byref(out)) == -1 and not out.value


def test_region_map_views_are_disjoint_and_inside_the_allocation():
    """every mode-specific tensor has a fixed region inside one allocation; views of
    ONE mode never overlap each other; TP and EP views of an object are one slot apart."""
    cfg = wl.get_config("fp8_graph").with_(L=2, E=8, H=256, I=1536, n_req=5, len_dist=("uniform", 1, 60))
    lens = wl.draw_seq_lens(cfg)
    sess = mb.Session(mb_config(cfg, lens))
    lay = sess.layout
    assert lay.base_bytes == lay.rank_stride_bytes * cfg.R
    for mode in (TP, EP):
        spans = []
        for r in range(cfg.R):
            for l in range(cfg.L):
                for t in range(8):
                    v = sess.view_desc(mode, r, l, t)
                    n = int(np.prod([v.shape[i] for i in range(v.ndim)])) * v.elem_bytes
                    assert v.offset % 256 == 0 and v.offset >= r * lay.rank_stride_bytes
                    assert v.offset + n <= (r + 1) * lay.rank_stride_bytes
                    spans.append((v.offset, v.offset + n))
        spans.sort()
        assert all(a[1] <= b[0] for a, b in zip(spans, spans[1:]))
    for r in range(cfg.R):
        for l in range(cfg.L):
            for t in range(3):
                a, b = sess.view_desc(TP, r, l, t), sess.view_desc(EP, r, l, t)
                assert b.offset - a.offset == lay.weight_slot_bytes
    # element counts: a rank holds 1/R of every object in both modes
    v_tp, v_ep = sess.view_desc(TP, 1, 0, 0), sess.view_desc(EP, 1, 0, 0)
    assert tuple(v_tp.shape[:3]) == (cfg.E, cfg.H, cfg.I // cfg.R) and tuple(v_ep.shape[:3]) == (cfg.E // cfg.R, cfg.H, cfg.I)
    d_tp, d_ep = sess.view_desc(TP, 1, 0, 2), sess.view_desc(EP, 1, 0, 2)
    assert tuple(d_tp.shape[:3]) == (cfg.E, cfg.I // cfg.R, cfg.H) and tuple(d_ep.shape[:3]) == (cfg.E // cfg.R, cfg.I, cfg.H)
    sess.close()


def test_scale_views_need_fp8():
    _, _, c = tiny_cfg()
    sess = mb.Session(c)
    with pytest.raises(mb.MoebiusError):
        sess.view_desc(TP, 0, 0, mb.T_GATE_SCALE)
    with pytest.raises(mb.MoebiusError):
        sess.view_desc(TP, 2, 0, mb.T_GATE)
    sess.close()


def test_capacity_failure_cancels_the_switch():
    """PAPER.md:211-213 / reading A16: the target mode cannot hold the requests -> E_CAPACITY, nothing
    is touched, and a retry with a request set that fits plans fine."""
    cfg = wl.get_config("tiny").with_(R=2, kv_heads=2)
    ep_page = cfg.page * cfg.kv_heads * cfg.head_dim * 2
    lens = np.array([64, 64, 64, 64, 64], np.int32)            # 4 pages each
    c = mb_config(cfg, lens, pool_bytes=10 * ep_page, max_pages=4, staging_cap_frac=0.9)
    sess = mb.Session(c)
    assert (sess.layout.pages_tp, sess.layout.pages_ep) == (20, 10)
    bt = np.arange(20, dtype=np.int32).reshape(5, 4)
    with pytest.raises(mb.MoebiusError) as e:                  # EP: 3 requests x 4 pages = 12 > 10 on one rank
        sess.plan(EP, lens, None, bt, from_mode=TP)
    assert e.value.status == -2
    ok = sess.plan(EP, lens[:4], None, bt[:4], from_mode=TP)   # the retry
    owner, _ = sess.block_tables(ok, 4)
    assert sorted(np.bincount(owner, minlength=2)) == [2, 2]
    sess.free_plan(ok)
    sess.close()


def test_tp_capacity_failure():
    """EP -> TP when the shared TP table cannot hold every request (replicated heads: G < R)."""
    cfg = wl.get_config("tiny").with_(R=4, E=8, I=64, kv_heads=2)     # G = 2: an EP page = 2 TP pages
    ep_page = cfg.page * cfg.kv_heads * cfg.head_dim * 2
    lens = np.array([64, 64, 64, 64], np.int32)                      # 16 TP pages needed
    c = mb_config(cfg, lens, pool_bytes=6 * ep_page, max_pages=4, staging_cap_frac=0.9)    # pages_ep 6, pages_tp 12
    sess = mb.Session(c)
    assert (sess.layout.pages_tp, sess.layout.pages_ep) == (12, 6)
    owner = np.arange(4, dtype=np.int32)
    bt = np.tile(np.arange(4, dtype=np.int32), (4, 1))
    with pytest.raises(mb.MoebiusError) as e:
        sess.plan(TP, lens, owner, bt, from_mode=EP)
    assert e.value.status == -2
    sess.free_plan(sess.plan(TP, lens[:3], owner[:3], bt[:3], from_mode=EP))
    sess.close()


def test_plan_argument_errors():
    cfg, lens, c = tiny_cfg()
    sess = mb.Session(c)
    mp = c.max_pages_per_request
    bt = wl.random_page_tables(lens, None, cfg.R, sess.layout.pages_tp, cfg.page, mp, seed=3)
    with pytest.raises(mb.MoebiusError):     # same mode on both sides
        sess.plan(TP, lens, None, bt, from_mode=TP)
    with pytest.raises(mb.MoebiusError):     # EP source needs the owner vector
        sess.plan(TP, lens, None, bt, from_mode=EP)
    dup = bt.copy()
    dup[1, 0] = dup[0, 0]
    with pytest.raises(mb.MoebiusError):     # a source page listed twice
        sess.plan(EP, lens, None, dup, from_mode=TP)
    bad = bt.copy()
    bad[0, 0] = sess.layout.pages_tp
    with pytest.raises(mb.MoebiusError):     # page id out of range
        sess.plan(EP, lens, None, bad, from_mode=TP)
    sess.close()


def test_reshard_fails_loudly_without_a_bound_device():
    """No CPU fallback: an unbound context is E_STATE; without a CUDA device the call is E_CUDA."""
    cfg, lens, c = tiny_cfg()
    sess = mb.Session(c)
    mp = c.max_pages_per_request
    bt = wl.random_page_tables(lens, None, cfg.R, sess.layout.pages_tp, cfg.page, mp, seed=3)
    plan = sess.plan(EP, lens, None, bt, from_mode=TP)
    with pytest.raises(mb.MoebiusError) as e:
        mb.moebius_reshard(sess.ctx, plan, 0)
    assert e.value.status == -4
    import torch
    if not torch.cuda.is_available():
        # bind to (host) addresses: the call must stop at the CUDA runtime, before touching them
        lay = sess.layout
        al = lambda n: (int(n) + 255) // 256 * 256  # noqa: E731
        sizes = [al(lay.base_bytes), al(max(lay.staging_bytes, 256)), al(lay.desc_bytes), al(lay.table_bytes)]
        host = np.zeros(sum(sizes) + 256, np.uint8)
        p0 = al(host.ctypes.data)
        ptrs = [p0 + sum(sizes[:k]) for k in range(4)]
        mb.moebius_bind(sess.ctx, ptrs[0], ptrs[1], ptrs[2], ptrs[3], TP)
        with pytest.raises(mb.MoebiusError) as e:
            mb.moebius_reshard(sess.ctx, plan, 0)
        assert e.value.status == -5
        assert mb.moebius_active_mode(sess.ctx) == TP     # nothing switched
        assert not host.any()                             # nothing written
    sess.close()


def test_status_strings():
    assert mb.moebius_status_str(0) == "ok"
    for s in (-1, -2, -3, -4, -5):
        assert mb.moebius_status_str(s) not in ("ok", "unknown")
    assert mb.moebius_version() >= 1


def test_header_is_plain_c():
    """The boundary is a C ABI: include/moebius.h must compile as C99 (and as C++) on its own."""
    import subprocess
    hdr = os.path.join(ROOT, "include", "moebius.h")
    for args in (["gcc", "-std=c99", "-pedantic", "-Wall", "-Werror", "-fsyntax-only", "-x", "c"],
                 ["g++", "-std=c++17", "-Wall", "-Werror", "-fsyntax-only", "-x", "c++"]):
        r = subprocess.run(args + [hdr], capture_output=True, text=True)
        assert r.returncode == 0, r.stderr


def test_plain_c_client_links_and_runs(tmp_path):
    """tests/abi_client.c: a C99 program against include/moebius.h + libmoebius.so, host-only calls."""
    import subprocess
    exe = str(tmp_path / "abi_client")
    lib_dir = os.path.dirname(mb.lib_path())
    r = subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                        os.path.join(ROOT, "tests", "abi_client.c"), "-o", exe, "-L", lib_dir, "-lmoebius",
                        "-Wl,-rpath," + lib_dir], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    r = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.startswith("OK"), r.stdout + r.stderr
