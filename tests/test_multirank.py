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
