"""N > 1 is "replicas only" (BASELINE.json fixes one GPU and excludes collectives): the
only cross-rank logic is bench.py's aggregation (sum of bytes / max of time) and the rule that the
reference arm runs on rank 0 alone.  Both are covered here with world_size 2 on the gloo backend."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
times, amounts = bench.reduce_over_ranks([10.0 + 5 * rank, 100.0 - rank], [7.0 * (rank + 1)], world, "cpu")
json.dump({"rank": rank, "times": times, "amounts": amounts}, open(os.path.join(sys.argv[1], "rank%%d.json" %% rank), "w"))
dist.destroy_process_group()
""" % ROOT


def torchrun(args, port):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port)] + args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)


def test_reduce_over_ranks_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    r = torchrun([str(script), str(tmp_path)], 29611)
    assert r.returncode == 0, r.stderr[-2000:]
    res = [json.load(open(tmp_path / ("rank%d.json" % k))) for k in range(2)]
    assert sorted(x["rank"] for x in res) == [0, 1]
    for x in res:
        assert x["times"] == [15.0, 100.0]      # max over ranks
        assert x["amounts"] == [21.0]           # sum over ranks


def test_reference_arm_runs_on_rank0_only():
    r = torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--config", "tiny", "--steps", "1", "--warmup", "0"], 29612)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"] and d["value"] > 0


def test_product_arm_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    r = subprocess.run([sys.executable, "bench.py", "--steps", "1", "--warmup", "1"], capture_output=True, text=True, cwd=ROOT,
                       timeout=600)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)


# ---- rank-share form of a switch, host side, world_size 2 on gloo -----------

SHARE_WORKER = r"""
import os, sys, json, hashlib
sys.path.insert(0, %r); sys.path.insert(0, os.path.join(%r, "tests"))
import numpy as np
import torch, torch.distributed as dist
import workloads as wl
import paper_2606_26607_b200 as mb
from paper_2606_26607_b200 import multiproc
from harness import mb_config
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
cfg = wl.get_config("small").with_(L=2, H=128, I=256, n_req=30, len_dist=("uniform", 1, 200), seed=61)
lens = wl.draw_seq_lens(cfg)
sess = mb.Session(mb_config(cfg, lens, "tight", 0.5))          # host only: the planner
bt = wl.random_page_tables(lens, None, cfg.R, sess.layout.pages_tp, cfg.page, sess.cfg.max_pages_per_request, seed=7)
plan = sess.plan(mb.MOEBIUS_EP, lens, None, bt, from_mode=mb.MOEBIUS_TP)
# 1. every process builds the same plan
digest = hashlib.sha256(mb.moebius_plan_export(plan, 0).tobytes() + mb.moebius_plan_export(plan, 1).tobytes()
                        + mb.moebius_plan_export(plan, 3).tobytes()).digest()
all_d = [None] * world
dist.all_gather_object(all_d, digest)
# 2. the shares partition the plan, wave by wave; crossing bytes sum to the owner-changed bytes
lo, hi = multiproc.owned_ranks(cfg.R, world, rank)
n_waves = mb.moebius_plan_waves(plan)
mine = np.array([[mb.moebius_share_stats(plan, lo, hi, w)[k] for k in ("units", "read", "written", "cross")]
                 for w in range(n_waves)], dtype=np.int64)
tot = torch.from_numpy(mine.copy())
dist.all_reduce(tot)
stats = mb.moebius_plan_stats(plan).as_dict()
# 3. the fd exchange the arena mapping uses, with ordinary files standing in for the allocations
fds = {}
for r in range(lo, hi):
    f = os.open(os.path.join(sys.argv[1], "region%%d" %% r), os.O_CREAT | os.O_RDWR)
    os.write(f, b"rank-%%d" %% r)
    fds[r] = f
peers = multiproc.exchange_fds(fds, cfg.R, world, rank, sys.argv[1], timeout_s=60)
seen = {}
for r, fd in peers.items():
    os.lseek(fd, 0, os.SEEK_SET)
    seen[r] = os.read(fd, 64).decode()
    os.close(fd)
json.dump({"rank": rank, "same_plan": all(d == digest for d in all_d), "n_waves": n_waves,
           "units_total": int(tot[:, 0].sum()), "cross_total": int(tot[:, 3].sum()),
           "n_units": stats["n_units"], "moved": stats["w_moved"] + stats["kv_moved"],
           "every_wave_has_units": bool((tot[:, 0] > 0).all()), "seen": seen, "owned": [lo, hi]},
          open(os.path.join(sys.argv[1], "share%%d.json" %% rank), "w"))
dist.barrier()
dist.destroy_process_group()
""" % (ROOT, ROOT)


def test_rank_share_host_logic_world2(tmp_path):
    import shutil
    import tempfile
    script = tmp_path / "share_worker.py"
    script.write_text(SHARE_WORKER)
    tmp_path = type(tmp_path)(tempfile.mkdtemp(prefix="mb", dir="/tmp"))   # AF_UNIX paths are limited to 108 bytes
    r = torchrun([str(script), str(tmp_path)], 29613)
    assert r.returncode == 0, r.stderr[-3000:]
    res = sorted((json.load(open(tmp_path / ("share%d.json" % k))) for k in range(2)), key=lambda x: x["rank"])
    assert [x["owned"] for x in res] == [[0, 2], [2, 4]]
    for x in res:
        assert x["same_plan"] and x["n_waves"] > 2
        assert x["units_total"] == x["n_units"] and x["cross_total"] == x["moved"]
        assert x["every_wave_has_units"]
    assert res[0]["seen"] == {"2": "rank-2", "3": "rank-3"} and res[1]["seen"] == {"0": "rank-0", "1": "rank-1"}
    shutil.rmtree(str(tmp_path), ignore_errors=True)
