"""Two PROCESSES, one GPU: the whole multi-process machinery of the rank-share switch for real
 -- each process owns half of the ranks as its own
physical allocations, maps the other half from its peer (fds over a unix socket), plans the same
switch, and executes only its ranks' units, one launch per dependency wave with a gloo barrier in
between, storing into / loading from the peer's regions.  No kernel ever waits for another kernel
(the profiling guide's rule for one GPU): the ordering is the host barrier.  Every process then
reads the WHOLE unified buffer through its own mapping and compares it with the oracle."""
import json
import os
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r); sys.path.insert(0, os.path.join(%r, "tests"))
import numpy as np
import torch, torch.distributed as dist
import workloads as wl
import paper_2606_26607_b200 as mb
from paper_2606_26607_b200 import multiproc
from paper_2606_26607_b200.session import _RawCuda
from harness import EP, TP, OracleLayout, State, expected_target, mb_config, source_tables
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
torch.cuda.set_device(0)                       # both processes share the one GPU of this box
cfg = wl.get_config("small").with_(L=2, H=128, I=256, n_req=30, len_dist=("uniform", 1, 200), seed=61,
                                   w_orient=int(sys.argv[2]))
st = State(cfg, fill="tag")
sess = mb.Session(mb_config(cfg, st.lens, "tight", 0.5), device="cuda:0")   # side buffers of THIS process
lay = sess.layout
lo, hi = multiproc.owned_ranks(cfg.R, world, rank)
arena = mb.moebius_arena_create(sess.ctx, 0, lo, hi)
multiproc.exchange_arena(arena, cfg.R, world, rank, sys.argv[1])
base = torch.as_tensor(_RawCuda(mb.moebius_arena_base(arena), int(lay.base_bytes)), device="cuda:0")
mb.moebius_bind(sess.ctx, base.data_ptr(), sess.staging.data_ptr(), sess.desc.data_ptr(), sess.tables.data_ptr(), TP)
# source layout: every process uploads ONLY the regions of the ranks it owns
owner, bt = source_tables(st, sess, TP, "random")
image = np.full(lay.base_bytes, 0xA5, np.uint8)
OracleLayout(st, sess, TP, owner, bt).place(image)
s0, s1 = lo * lay.rank_stride_bytes, hi * lay.rank_stride_bytes
base[s0:s1].copy_(torch.from_numpy(image[s0:s1]))
torch.cuda.synchronize(); dist.barrier()
report = {"rank": rank, "owned": [lo, hi], "bad": [], "waves": [], "cross": []}
mode = TP
for k in range(2):
    to = EP if mode == TP else TP
    plan = sess.plan(to, st.lens, owner, bt, from_mode=mode)
    report["waves"].append(mb.moebius_plan_waves(plan))
    report["cross"].append(mb.moebius_share_stats(plan, lo, hi)["cross"])
    multiproc.switch(sess.ctx, plan, cfg.R, world, rank, dist.barrier, torch.cuda.current_stream().cuda_stream,
                     torch.cuda.synchronize)
    want_owner, want_bt = expected_target(st, sess, to)
    got = base.cpu().numpy()                    # ALL ranks, through this process's mapping
    report["bad"] += OracleLayout(st, sess, to, want_owner, want_bt).compare(got)[:3]
    t = sess.tables.cpu().numpy()
    report["bad"] += [] if (t[0] == to and np.array_equal(t[lay.tbl_bt_off:lay.tbl_bt_off + want_bt.size].reshape(want_bt.shape), want_bt)) else ["tables"]
    sess.free_plan(plan)
    owner, bt, mode = (want_owner if to == EP else None), want_bt, to
    dist.barrier()
json.dump(report, open(os.path.join(sys.argv[1], "mp%%d.json" %% rank), "w"))
del base
sess.base = None
torch.cuda.synchronize(); dist.barrier()
mb.moebius_arena_destroy(arena)
dist.destroy_process_group()
""" % (ROOT, ROOT)


@pytest.mark.parametrize("orient", [0, 1])
def test_two_processes_share_one_switch(tmp_path, orient):
    assert torch.cuda.is_available()
    import shutil
    import tempfile
    script = tmp_path / "mp_worker.py"
    script.write_text(WORKER)
    tmp_path = type(tmp_path)(tempfile.mkdtemp(prefix="mb", dir="/tmp"))   # AF_UNIX paths are limited to 108 bytes
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(29621 + orient), str(script), str(tmp_path), str(orient)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, (r.stdout + r.stderr)[-3000:]
    res = sorted((json.load(open(tmp_path / ("mp%d.json" % k))) for k in range(2)), key=lambda x: x["rank"])
    assert [x["owned"] for x in res] == [[0, 2], [2, 4]]
    for x in res:
        assert not x["bad"], x["bad"]
        assert x["waves"][0] > 2                 # tight pool from random tables: real dependency rounds
        assert all(c > 0 for c in x["cross"])    # each process really moved bytes into / out of its peer's regions
    shutil.rmtree(str(tmp_path), ignore_errors=True)
