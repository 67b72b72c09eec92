#!/usr/bin/env python
"""bench.py -- per-switch time and effective GB/s of the TP<->EP reshard on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config qwen3_235b] [--impl reference]

A STEP is one round trip of the whole hot path, TP->EP then EP->TP, over one synthetic request set
(plan, request ownership, block tables, descriptors, expert-weight relayout, KV
relayout, publish).  `value` = owner-changed bytes of both switches / device time (inputs resident
in HBM, plans built before the timed region, CUDA events round K steps of `moebius_reshard`).
`e2e` = the same metric through the C ABI starting from HOST inputs (seq_lens, owners and block
tables in host memory): moebius_plan + moebius_reshard (work-list and table upload) for both switches
of the step -- the second is planned while the first runs, moebius_reshard only enqueues -- + a
device->host read-back of the published tables, every step, timed on the host round a synchronize.  The
weights and the KV cache are resident by the definition of the method (one
resident copy at fixed addresses), so they are not re-uploaded per step.
N > 1: independent replicas, one per GPU, no collective; value is the
sum over ranks / max time over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

METRIC = "reshard_owner_changed_GBps_per_TP<->EP_round_trip"
UNIT = "GB/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="qwen3_235b")
    ap.add_argument("--impl", default="moebius", choices=["moebius", "reference"])
    ap.add_argument("--pool", default="roomy", choices=["roomy", "tight"])
    ap.add_argument("--launch", default="", help="ctas_per_sm,threads,unit_kb (tuning)")
    ap.add_argument("--layers", type=int, default=0, help="override L (profiling captures only; named in config.workload)")
    ap.add_argument("--staging-cap-frac", type=float, default=0.024,
                    help="cap on spare slot + staging as a fraction of resident bytes (0 = library default)")
    ap.add_argument("--n-req", type=int, default=-1, help="override the number of live requests (experiments; named in config.workload)")
    ap.add_argument("--tma", default="", help="enable,pipes,stage_kb (tuning; default: library defaults)")
    ap.add_argument("--ring", default="", help="ring_kb,max_loads of the pipes' rings (tuning; after --tma)")
    ap.add_argument("--l2", default="", help="load,store L2 cache-hint policy of the TMA operations (tuning)")
    ap.add_argument("--kv-rounds", type=int, default=0, help="max dependent KV rounds before chains are cut by staging (tuning)")
    ap.add_argument("--xt-mode", type=int, default=-1, help="weight tensor-map box side: 0 EP views, 1 TP views (tuning / A-B)")
    ap.add_argument("--chain-bands", action="store_true", help="banded weight chain: links overlap half by half (tuning / A-B; off by default)")
    ap.add_argument("--kv-slice", type=int, default=0, help="smallest KV slice interleaved with the weight chain, in units (tuning)")
    ap.add_argument("--w-orient", type=int, default=0, choices=[0, 1],
                    help="0: gate,up [E,H,I], down [E,I,H] (BASELINE.json, the headline); 1: the paper's W13 [E,2I,H], W2 [E,H,I] (named in config.workload)")
    ap.add_argument("--w-inplace", action="store_true",
                    help="force shift 0: EP and TP views alias the same bytes, every object takes the in-place path (named in config.workload)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-naive", action="store_true", help="skip timing the staged comparison path (PAPER.md Table 1)")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="default run only: skip timing configs 3, 5, 2 and the tight-pool variant after config 4")
    ap.add_argument("--profile-region", action="store_true",
                    help="cudaProfilerStart/Stop round warm-up + timed steps (ncu --profile-from-start off skips the fill)")
    ap.add_argument("--cpu-sample-requests", type=int, default=48)
    return ap.parse_args()


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


KERNEL_SOURCES = ("paper_2606_26607_b200/csrc/moebius_cuda.cu", "paper_2606_26607_b200/csrc/moebius_units.h")


def kernel_sha16():
    """First 16 hex digits of sha256 over the kernel's source files: ties a committed ncu figure to the
    kernel it was measured on."""
    import hashlib
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        h.update(open(os.path.join(ROOT, f), "rb").read())
    return h.hexdigest()[:16]


def committed_traffic(config_name):
    """(traffic, source): DRAM bytes per launch of the reshard kernel (dram__bytes_read.sum +
    dram__bytes_write.sum) from the committed ncu capture of this config, with where it came from.
    None when there is no capture or when the kernel sources have changed since it was taken."""
    p = os.path.join(ROOT, "profiles", "traffic_%s.txt" % config_name)
    if not os.path.exists(p):
        return None, "no ncu capture committed for this config"
    kv = {}
    for line in open(p):
        if "=" in line and not line.startswith("#"):
            k, v = line.strip().split("=", 1)
            kv[k] = v
    if kv.get("kernel_sha16") != kernel_sha16():
        return None, "stale: %s was captured on kernel %s, HEAD's kernel is %s" % (
            os.path.relpath(p, ROOT), kv.get("kernel_sha16"), kernel_sha16())
    return float(kv["traffic_bytes_per_launch"]), "%s (ncu, %s, commit %s)" % (
        kv.get("capture", os.path.relpath(p, ROOT)), kv.get("command", "see profiles/README.md"), kv.get("commit", "?"))


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 6:
                    self.rows.append(f)
            except Exception:
                pass
            time.sleep(0.05)

    def summary(self):
        self.stop_flag = True
        self.join(timeout=6)
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "reasons": reasons,
                "samples": len(self.rows)}


# ---- the oracle, timed as it stands (cpu_baseline leg and --impl reference) ---------------------------

def oracle_sample(cfg, n_sample_req, layer=0, seed=0):
    """Logical state of the bounded sample: ONE layer of the expert weights (gate, up, down, all E
    experts) and that layer's K and V of the first `n_sample_req` requests of the workload."""
    rng = np.random.default_rng((seed, layer))
    dt = {"bf16": np.uint16, "fp32": np.float32, "fp8_e4m3_b128": np.uint8}[cfg.w_dtype]
    W = {}
    for kind in cfg.w_kinds:
        shape = wl.weight_shape(cfg, kind)
        if dt == np.float32:
            W[kind] = rng.standard_normal(shape, dtype=np.float32)
        else:   # opaque bit patterns: generation cost is excluded from the timing anyway
            W[kind] = rng.integers(0, np.iinfo(dt).max, size=shape, dtype=dt, endpoint=True)
    lens = wl.draw_seq_lens(cfg)[:n_sample_req]
    KV = [{i: wl.gen_kv_request(cfg, layer, kvi, i, int(n)) for i, n in enumerate(lens)} for kvi in range(2)]
    return W, lens, KV


def oracle_round_trip(cfg, W, lens, KV, pool_bytes):
    """One round trip as the oracle computes it: the EP layout, then the TP layout, each built from
    the logical tensors (oracle/: weights.py, kv.py).  Returns owner-changed bytes of the sample."""
    import oracle
    R, Hkv, D, pg = cfg.R, cfg.kv_heads, cfg.head_dim, cfg.page
    hpr = max(1, Hkv // R)
    ep_page = pg * Hkv * D * cfg.kv_elem_bytes
    pages_ep = pool_bytes // ep_page
    pages_tp = pages_ep * min(Hkv, R)
    mp = int(max([1] + [oracle.pages_needed(n, pg) for n in lens]))
    assert hpr >= 1
    # TP -> EP
    owner = oracle.partition_requests(lens, R)
    bt_ep = oracle.canonical_block_tables(lens, owner, "ep", pages_ep, pg, mp)
    for r in range(R):
        for kind in cfg.w_kinds:
            oracle.ep_weight_view(W[kind], r, R)
        for kvi in range(2):
            oracle.ep_pool_image(KV[kvi], lens, owner, bt_ep, r, Hkv, D, pg, pages_ep)
    # EP -> TP
    bt_tp = oracle.canonical_block_tables(lens, None, "tp", pages_tp, pg, mp)
    for r in range(R):
        for kind in cfg.w_kinds:
            oracle.tp_weight_view(W[kind], kind, r, R)
        for kvi in range(2):
            oracle.tp_pool_image(KV[kvi], lens, bt_tp, r, R, Hkv, D, pg, pages_tp)
    return owner


def oracle_sample_moved(cfg, lens, owner):
    """Owner-changed bytes of one round trip over the sample (oracle/accounting.py), outside the timing."""
    import oracle
    moved = 0
    for d in ("tp2ep", "ep2tp"):
        moved += oracle.weight_bytes(cfg.R, 1, cfg.E, cfg.H, cfg.I, cfg.w_elem_bytes, d)["moved"]
        moved += oracle.kv_bytes(lens, owner, cfg.R, 1, cfg.kv_heads, cfg.head_dim, cfg.kv_elem_bytes, d)["moved"]
    return moved


def _sample_text(cfg, n_lens, layers):
    return ("layer%s %s of %d: %s of all %d experts + K and V pools of the first %d of %d requests; "
            "one TP->EP->TP round trip per step" % ("s" if len(layers) > 1 else "", ",".join(str(l) for l in layers), cfg.L,
                                                    "/".join(cfg.w_kinds), cfg.E, n_lens, cfg.n_req))


def time_oracle(cfg, n_sample_req, steps, warmup, pool_bytes, layer=0):
    """Single-thread leg: the oracle as it stands on one layer's sample, in this process."""
    W, lens, KV = oracle_sample(cfg, n_sample_req, layer)
    for _ in range(warmup):
        oracle_round_trip(cfg, W, lens, KV, pool_bytes)
    t0 = time.perf_counter()
    for _ in range(steps):
        owner = oracle_round_trip(cfg, W, lens, KV, pool_bytes)
    dt = time.perf_counter() - t0
    moved = steps * oracle_sample_moved(cfg, lens, owner)
    return {"value": moved / dt / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": _sample_text(cfg, len(lens), [layer]), "seconds": dt, "ms_per_step": dt / steps * 1e3,
            "moved_bytes": moved}


def _oracle_worker(cfg, n_sample_req, pool_bytes, layer, ready, go, out):
    """One process of the per-core leg: layers are independent, so worker w
    builds the views of its own layer.  Generation happens before the common start signal."""
    W, lens, KV = oracle_sample(cfg, n_sample_req, layer)
    ready.put(layer)
    go.wait()
    t0 = time.perf_counter()
    owner = oracle_round_trip(cfg, W, lens, KV, pool_bytes)
    t1 = time.perf_counter()
    out.put((layer, t0, t1, oracle_sample_moved(cfg, lens, owner)))


def time_oracle_per_core(cfg, n_sample_req, pool_bytes, host_cores):
    """Per-core leg: one oracle process per host core, each on its own layer (at most L processes, and
    no more than the host memory allows: one layer of logical state + its views per process)."""
    import multiprocessing as mp
    layer_bytes = sum(int(np.prod(wl.weight_shape(cfg, k))) for k in cfg.w_kinds) * cfg.w_elem_bytes
    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:
        avail = 32 << 30
    by_mem = max(1, int(avail * 0.6 // max(1, int(layer_bytes * 1.6))))
    n = max(1, min(host_cores, cfg.L, by_mem, 16))
    ctx = mp.get_context("spawn")     # this process holds a CUDA context: never fork it
    ready, out, go = ctx.Queue(), ctx.Queue(), ctx.Event()
    procs = [ctx.Process(target=_oracle_worker, args=(cfg, n_sample_req, pool_bytes, l, ready, go, out)) for l in range(n)]
    for p in procs:
        p.start()

    def take(q, deadline_s=600):      # a worker that died must not leave the bench waiting
        t_end = time.time() + deadline_s
        while True:
            try:
                return q.get(timeout=1.0)
            except Exception:
                if any(p.exitcode not in (None, 0) for p in procs) or time.time() > t_end:
                    for p in procs:
                        if p.is_alive():
                            p.terminate()
                    raise RuntimeError("an oracle worker exited early")

    for _ in procs:
        take(ready)
    go.set()
    res = [take(out) for _ in procs]
    for p in procs:
        p.join(timeout=60)
    t0, t1 = min(r[1] for r in res), max(r[2] for r in res)    # perf_counter is system-wide on Linux
    moved = sum(r[3] for r in res)
    return {"value": moved / (t1 - t0) / 1e9, "unit": UNIT, "cores": n, "kind": "oracle",
            "sample": _sample_text(cfg, min(n_sample_req, cfg.n_req), list(range(n))) + "; one process per layer, concurrently",
            "seconds": t1 - t0}


def cpu_baseline(cfg, n_sample_req, pool_bytes, per_core=True):
    """the oracle timed once single-threaded and once with one process per host
    core over layers; `cores` = what the reported leg actually used, `host_cores` = sched_getaffinity."""
    host_cores = len(os.sched_getaffinity(0))
    one = time_oracle(cfg, n_sample_req, 1, 0, pool_bytes)
    out = {"value": one["value"], "unit": UNIT, "cores": 1, "kind": "oracle", "sample": one["sample"],
           "host_cores": host_cores, "single_thread": {"value": one["value"], "cores": 1, "seconds": one["seconds"]}}
    if per_core and host_cores > 1:
        try:
            many = time_oracle_per_core(cfg, n_sample_req, pool_bytes, host_cores)
            out.update({"value": many["value"], "cores": many["cores"], "sample": many["sample"],
                        "per_core": {"value": many["value"], "cores": many["cores"], "seconds": many["seconds"]}})
        except Exception as e:      # a reported baseline must not take the bench line down
            out["per_core"] = {"error": repr(e)[:200]}
    return out


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores (tier framing: the oracle is the reference arm)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = wl.get_config(args.config)
    pool = wl.kv_pool_bytes(cfg, wl.draw_seq_lens(cfg), args.pool)
    steps, warmup = max(1, min(args.steps, 3)), min(args.warmup, 1)
    r = time_oracle(cfg, args.cpu_sample_requests, steps, warmup, pool)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
            "config": {"workload": cfg.name, "sample": r["sample"]},
            "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
                             "sample": r["sample"], "host_cores": len(os.sched_getaffinity(0))},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---- the product arm ----------------------------------------------------------------------------------

def fill_device(sess, cfg, mb, torch):
    """Synthetic resident state (BASELINE.json: experts ~N(0,0.02), KV ~N(0,1)), generated on the
    device with a seeded generator: only memory plumbing, the values do not affect the timing."""
    g = torch.Generator(device=sess.device)
    g.manual_seed(cfg.seed)
    for r in range(cfg.R):
        for l in range(cfg.L):
            for t in ((mb.T_GATE, mb.T_UP, mb.T_DOWN) if cfg.w_orient == 0 else (mb.T_W13, mb.T_W2)):
                v = sess.view(mb.MOEBIUS_TP, r, l, t)
                if v.dtype == torch.int16:
                    v.view(torch.bfloat16).normal_(0.0, 0.02, generator=g)
                elif v.dtype == torch.float32:
                    v.normal_(0.0, 0.02, generator=g)
                else:
                    v.random_(0, 255, generator=g)
            for t in (mb.T_KPOOL, mb.T_VPOOL):
                sess.view(mb.MOEBIUS_TP, r, l, t).view(torch.bfloat16).normal_(0.0, 1.0, generator=g)


def init_device():
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device; there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    return world, rank, local, dev


def run_moebius(args, env, config_name, pool_policy, cap_frac, steps, warmup, full=True, overrides=None):
    """Times one workload.  full=False (the other_configs entries): kernel times only -- no D2D
    comparison copy, no e2e loop."""
    import torch
    import torch.distributed as dist

    import paper_2606_26607_b200 as mb   # fails loudly if libmoebius.so is missing: no CPU fallback

    world, rank, local, dev = env
    cfg = wl.get_config(config_name)
    if overrides:
        cfg = cfg.with_(name="%s[%s]" % (cfg.name, ",".join("%s=%s" % kv for kv in sorted(overrides.items()))), **overrides)
    if args.layers:
        cfg = cfg.with_(L=args.layers, name="%s[L=%d]" % (cfg.name, args.layers))
    if args.w_orient and not overrides:
        cfg = cfg.with_(w_orient=1, name="%s[w_orient=1]" % cfg.name)
    if args.w_inplace and not overrides:
        cfg = cfg.with_(w_inplace=1, name="%s[w_inplace=1]" % cfg.name)
    lens = wl.draw_seq_lens(cfg)
    pool = wl.kv_pool_bytes(cfg, lens, pool_policy)
    if args.n_req >= 0:
        lens = lens[:args.n_req]
        cfg = cfg.with_(n_req=args.n_req, name="%s[n_req=%d]" % (cfg.name, args.n_req))
    mp = int(max([1] + [(int(x) + cfg.page - 1) // cfg.page for x in lens]))
    c = mb.make_config(R=cfg.R, L=cfg.L, E=cfg.E, H=cfg.H, I=cfg.I, w_dtype=cfg.w_dtype, kv_heads=cfg.kv_heads,
                       head_dim=cfg.head_dim, page_tokens=cfg.page, kv_pool_bytes_per_rank_layer=pool,
                       max_requests=max(len(lens), 1), max_pages_per_request=mp, staging_cap_bytes=0,
                       w_orient=cfg.w_orient, w_inplace=cfg.w_inplace)
    probe = mb.Session(c)
    resident = probe.layout.resident_bytes
    probe.close()
    c.staging_cap_bytes = int(cap_frac * resident)   # BASELINE.json: cap at ~2.4% of resident bytes
    sess = mb.Session(c, device=dev)
    lay = sess.layout
    if args.launch:
        a, b, u = (int(x) for x in args.launch.split(","))
        mb.moebius_set_launch(sess.ctx, a, b, u)
    if args.tma:
        a, b, u = (int(x) for x in args.tma.split(","))
        mb.moebius_set_tma(sess.ctx, a, b, u)
    if args.ring:
        a, b = (int(x) for x in args.ring.split(","))
        mb.moebius_set_ring(sess.ctx, a, b)
    if args.l2:
        a, b = (int(x) for x in args.l2.split(","))
        mb.moebius_set_l2_policy(sess.ctx, a, b)
    if args.kv_rounds:
        mb.moebius_set_kv_rounds(sess.ctx, args.kv_rounds)
    if args.kv_slice:
        mb.moebius_set_kv_slice(sess.ctx, args.kv_slice)
    if args.chain_bands:
        mb.moebius_set_chain_bands(sess.ctx, True)
    if args.xt_mode >= 0:
        mb.moebius_set_xt_mode(sess.ctx, args.xt_mode)
    fill_device(sess, cfg, mb, torch)
    TP, EP = mb.MOEBIUS_TP, mb.MOEBIUS_EP
    n = len(lens)
    stream = torch.cuda.current_stream()

    # state: TP with seeded random page tables (reading A8)
    bt0 = wl.random_page_tables(lens, None, cfg.R, lay.pages_tp, cfg.page, mp, seed=cfg.seed)

    def switch(to, owner, bt, frm):
        t0 = time.perf_counter()
        plan = sess.plan(to, lens, owner, bt, from_mode=frm)
        t1 = time.perf_counter()
        sess.reshard(plan)
        new_owner, new_bt = sess.block_tables(plan, n)
        return plan, (new_owner if to == EP else None), new_bt, (t1 - t0) * 1e3

    mb.moebius_set_timing(sess.ctx, True)
    if args.profile_region:
        torch.cuda.synchronize()
        torch.cuda.cudart().cudaProfilerStart()
    # warm-up: W round trips (the first one starts from the random tables)
    owner, bt, mode = None, bt0, TP
    first_ms = {}
    for w in range(max(warmup, 1)):
        for to in (EP, TP):
            plan, owner, bt, _ = switch(to, owner, bt, mode)
            if w == 0:
                fs = mb.moebius_plan_stats(plan).as_dict()
                first_ms["tp2ep" if to == EP else "ep2tp"] = {
                    "kernel_ms": mb.moebius_last_kernel_ms(sess.ctx), "kv_rounds": fs["n_kv_rounds"],
                    "kv_staged": fs["n_kv_staged"], "pool_groups": fs["n_pool_groups"], "segments": fs["n_segments"]}
            sess.free_plan(plan)
            mode = to
    torch.cuda.synchronize()
    # steady state: TP with canonical tables; both plans built once, before the timed region
    plan_t2e, owner_ep, bt_ep, plan_ms_t2e = switch(EP, None, bt, TP)
    plan_e2t, _, bt_tp, plan_ms_e2t = switch(TP, owner_ep, bt_ep, EP)
    assert np.array_equal(bt_tp, bt)
    torch.cuda.synchronize()
    st_t2e = mb.moebius_plan_stats(plan_t2e).as_dict()
    st_e2t = mb.moebius_plan_stats(plan_e2t).as_dict()

    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        sess.reshard(plan_t2e)
        sess.reshard(plan_e2t)
    e1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    dev_ms = e0.elapsed_time(e1)
    if args.profile_region and (not full or args.no_naive):
        torch.cuda.cudart().cudaProfilerStop()
    hist = mb.moebius_kernel_ms_history(sess.ctx, 64)[-2 * steps:]
    k_t2e, k_e2t = hist[0::2], hist[1::2]
    # context: a plain device-to-device copy of a weight slot on this box, now (read + write bytes)
    d2d = None
    if cfg.R > 1 and full:
        n_copy = int(min(lay.weight_slot_bytes * (3 * cfg.L), 8 << 30)) // 256 * 256
        t0_id = mb.T_GATE if cfg.w_orient == 0 else mb.T_W13
        a0 = sess.view_desc(TP, 0, 0, t0_id).offset
        a1 = sess.view_desc(TP, cfg.R - 1, 0, t0_id).offset
        src, dst = sess.base[a0:a0 + n_copy], sess.base[a1:a1 + n_copy]
        keep = dst.clone()
        best = None
        for _ in range(5):
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            c0.record(stream)
            dst.copy_(src)
            c1.record(stream)
            torch.cuda.synchronize()
            ms = c0.elapsed_time(c1)
            best = ms if best is None else min(best, ms)
        dst.copy_(keep)
        del keep
        torch.cuda.synchronize()
        d2d = {"bytes": n_copy, "ms_best_of_5": best, "GBps_read_plus_write": 2 * n_copy / best / 1e6}

    sess.free_plan(plan_t2e)     # their pinned upload images go back to the context's pool
    sess.free_plan(plan_e2t)
    if not full:
        clocks = sampler.summary()
        sess.close()
        return {k: v for k, v in locals().items() if not isinstance(v, (torch.Tensor, mb.Session))}
    # e2e: host inputs -> plan -> reshard (uploads) -> device->host read-back of the published tables
    host_tables = torch.empty(lay.table_bytes // 4, dtype=torch.int32, pin_memory=True)
    tbl_n = lay.tbl_bt_off + n * mp
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    owner, bt_cur, mode = None, bt, TP
    h2d = d2h = 0
    plan_ms = []
    for _ in range(steps):
        # moebius_reshard only enqueues: the second switch of the step is planned on the host while the
        # first one runs on the device (its inputs are the first plan's tables, known on the host)
        live = []
        for to in (EP, TP):
            plan, owner, bt_cur, pms = switch(to, owner, bt_cur, mode)
            s = mb.moebius_plan_stats(plan)
            h2d += s.desc_upload_bytes + s.table_upload_bytes
            plan_ms.append(pms)
            live.append(plan)
            mode = to
        host_tables[:tbl_n].copy_(sess.tables[:tbl_n], non_blocking=True)   # the step's result
        torch.cuda.synchronize()
        assert int(host_tables[0]) == TP and int(host_tables[1]) == n
        d2h += tbl_n * 4
        for plan in live:
            sess.free_plan(plan)
    e2e_s = time.perf_counter() - t0
    clocks = sampler.summary()
    # the staged comparison path of PAPER.md Table 1 (permute -> exchange -> scatter through a staging
    # buffer), timed on the same resident state right after the fused kernel: context, not the metric
    naive = None
    if not args.no_naive:
        try:
            naive = {"tp2ep_ms": [], "ep2tp_ms": []}
            scratch = None
            for _ in range(2):
                for to in (EP, TP):
                    plan = sess.plan(to, lens, owner, bt_cur, from_mode=mode)
                    need = mb.moebius_naive_scratch_bytes(sess.ctx, plan)
                    if scratch is None or scratch.numel() < need + 256:
                        scratch = None
                        scratch = torch.empty(int(need * 1.05) + 4096, dtype=torch.uint8, device=dev)
                    off = (-scratch.data_ptr()) % 256
                    ns = mb.moebius_reshard_naive(sess.ctx, plan, scratch.data_ptr() + off, scratch.numel() - off, stream.cuda_stream)
                    torch.cuda.synchronize()
                    naive["tp2ep_ms" if to == EP else "ep2tp_ms"].append(mb.moebius_last_kernel_ms(sess.ctx))
                    naive["tp2ep" if to == EP else "ep2tp"] = ns
                    new_owner, bt_cur = sess.block_tables(plan, n)
                    owner = new_owner if to == EP else None
                    sess.free_plan(plan)
                    mode = to
            del scratch
        except Exception as e:      # context only: never take the bench line down
            naive = {"error": repr(e)[:300]}
        if args.profile_region:
            torch.cuda.synchronize()
            torch.cuda.cudart().cudaProfilerStop()
    sess.close()
    # no tensor and no session leaves this function: the device buffers go back to torch before the next
    # workload is built
    return {k: v for k, v in locals().items() if not isinstance(v, (torch.Tensor, mb.Session))}


def reduce_over_ranks(times_ms, amounts, world, device):
    """Replicas only: every rank runs the same independent job on its own GPU, so the
    whole-job figure is (sum over ranks of the bytes) / (max over ranks of the time).  No data-path
    collective exists; these two all-reduces of a few scalars happen after the timed region."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    b = torch.tensor(list(amounts), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(b, op=dist.ReduceOp.SUM)
    return [float(x) for x in t], [float(x) for x in b]


def direction_summary(st, ms_list, peak):
    avg = float(sum(ms_list) / max(len(ms_list), 1))
    med = float(sorted(ms_list)[len(ms_list) // 2]) if ms_list else None
    traffic = st["w_read"] + st["w_relocated"] + st["kv_read"] + st["kv_relocated"]
    moved = st["w_moved"] + st["kv_moved"]
    return {"kernel_ms_avg": avg, "kernel_ms_min": min(ms_list) if ms_list else None, "kernel_ms_median": med,
            "moved_bytes": moved, "algorithmic_traffic_bytes": traffic,
            "effective_GBps": moved / avg / 1e6 if avg else None,
            "traffic_GBps": traffic / avg / 1e6 if avg else None,
            "frac_strict_vs_8TBps": 2 * moved / (avg * 1e-3) / 8e12 if avg else None,
            "frac_traffic_vs_measured": traffic / avg / 1e6 / peak if avg else None,
            "units": st["n_units"], "segments": st["n_segments"], "kv_moves": st["n_kv_moves"],
            "kv_rounds": st["n_kv_rounds"], "kv_staged": st["n_kv_staged"]}


def split_history(hist):
    m = len(hist) // 2 * 2
    hist = hist[len(hist) - m:]
    return hist[0::2], hist[1::2]


# The parity-test configs of BASELINE.json and the cache-nearly-full variant of config 4, timed after the
# headline workload in the default run so that the driver's record carries them too.
OTHER_CONFIGS = (("qwen3_30b", "qwen3_30b", "roomy", 0.024, None), ("fp8_graph", "fp8_graph", "roomy", 0.024, None),
                 ("small", "small", "roomy", 0.024, None), ("qwen3_235b_tight_pool", "qwen3_235b", "tight", 0.024, None),
                 # the paper's own orientation: config 4 inside the cap with two spare slots; config 5
                 # only with one, so its W13 objects take the in-place path (S2: dependency waves, parked blocks)
                 ("qwen3_235b_paper_orient", "qwen3_235b", "roomy", 0.024, {"w_orient": 1}),
                 ("fp8_graph_paper_orient_in_place", "fp8_graph", "roomy", 0.024, {"w_orient": 1}),
                 # config 4 with NO spare slot at all: EP and TP views alias the same bytes (shift 0), every object
                 # is permuted in place through the staging buffer, under a cap of 1.2 % of resident
                 ("qwen3_235b_aliased_in_place", "qwen3_235b", "roomy", 0.012, {"w_inplace": 1}))


def other_config_entry(r, peak):
    k_t2e, k_e2t = split_history(r["hist"])
    a, b = direction_summary(r["st_t2e"], k_t2e, peak), direction_summary(r["st_e2t"], k_e2t, peak)
    lay = r["lay"]
    return {"workload": r["cfg"].name, "kv_pool": r["pool_policy"], "steps": r["steps"],
            "tp2ep_ms": a["kernel_ms_avg"], "ep2tp_ms": b["kernel_ms_avg"],
            "traffic_GBps": [a["traffic_GBps"], b["traffic_GBps"]],
            "effective_GBps": [a["effective_GBps"], b["effective_GBps"]],
            "frac_strict": [a["frac_strict_vs_8TBps"], b["frac_strict_vs_8TBps"]],
            "frac_traffic_vs_measured": [a["frac_traffic_vs_measured"], b["frac_traffic_vs_measured"]],
            "kv_rounds": [a["kv_rounds"], b["kv_rounds"]], "kv_staged": [a["kv_staged"], b["kv_staged"]],
            "first_switch_from_random_tables": r["first_ms"],
            "w_shift_slots": lay.w_shift_slots, "w_waves": [r["st_t2e"]["n_w_waves"], r["st_e2t"]["n_w_waves"]],
            "w_parked_blocks": [r["st_t2e"]["n_w_parked"], r["st_e2t"]["n_w_parked"]],
            "resident_GB": lay.resident_bytes / 1e9,
            "spare_plus_staging_frac": (lay.weight_spare_bytes + lay.staging_bytes) / lay.resident_bytes,
            "staging_cap_frac": r["cap_frac"], "ms_per_step": r["dev_ms"] / r["steps"], "clocks": r["clocks"]}


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    import torch
    import torch.distributed as dist
    env = init_device()
    r = run_moebius(args, env, args.config, args.pool, args.staging_cap_frac, args.steps, max(args.warmup, 1))
    world, rank, cfg, steps = r["world"], r["rank"], r["cfg"], args.steps
    st_t2e, st_e2t = r["st_t2e"], r["st_e2t"]
    moved_step = st_t2e["w_moved"] + st_t2e["kv_moved"] + st_e2t["w_moved"] + st_e2t["kv_moved"]
    (dev_ms, e2e_ms), (moved_all,) = reduce_over_ranks([r["dev_ms"], r["e2e_s"] * 1e3], [float(moved_step)], world, r["dev"])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    k_t2e, k_e2t = split_history(r["hist"])
    avg = lambda x: float(sum(x) / max(len(x), 1))  # noqa: E731
    peak, peak_src = measured_peak()
    d_t2e, d_e2t = direction_summary(st_t2e, k_t2e, peak), direction_summary(st_e2t, k_e2t, peak)
    # roofline of the dominant (only) kernel: algorithmic bytes per launch / average launch duration
    alg = (d_t2e["algorithmic_traffic_bytes"] + d_e2t["algorithmic_traffic_bytes"]) / 2
    k_ms = avg(k_t2e + k_e2t)
    achieved = alg / k_ms / 1e6
    lay = r["lay"]
    traffic, traffic_src = committed_traffic(cfg.name) if args.pool == "roomy" else (None, "no capture for this pool policy")
    line = {
        "metric": METRIC, "value": moved_all * steps / dev_ms / 1e6, "unit": UNIT, "n_gpus": world, "steps": steps,
        "warmup": max(args.warmup, 1), "ms_per_step": dev_ms / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": cfg.name, "R": cfg.R, "L": cfg.L, "E": cfg.E, "H": cfg.H, "I": cfg.I,
                   "w_dtype": cfg.w_dtype, "kv_heads": cfg.kv_heads, "head_dim": cfg.head_dim, "page": cfg.page,
                   "n_req": cfg.n_req, "live_tokens": int(r["lens"].sum()), "kv_pool": args.pool,
                   "resident_GB": lay.resident_bytes / 1e9, "spare_plus_staging_frac":
                   (lay.weight_spare_bytes + lay.staging_bytes) / lay.resident_bytes,
                   "step": "one TP->EP + one EP->TP switch", "l2": "working set >> L2 (126 MB); no flush needed",
                   "parallelism": "replicas only" if world > 1 else "1 GPU, R logical ranks as regions"},
        "tp2ep": d_t2e, "ep2tp": d_e2t,
        "first_switch_from_random_tables": r["first_ms"],
        "d2d_copy_same_box": r["d2d"],
        "plan_ms": {"tp2ep": r["plan_ms_t2e"], "ep2tp": r["plan_ms_e2t"], "e2e_avg": avg(r["plan_ms"])},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "frac_note": "vs the measured D2D copy rate of this pool (a copy, not a physical peak); "
                                  "the strict fraction 2*moved/(t*8 TB/s) is in tp2ep/ep2tp.frac_strict_vs_8TBps",
                     "traffic": traffic, "traffic_source": traffic_src, "kernel_sha16": kernel_sha16(),
                     "peak_source": peak_src,
                     "kernel": "moebius_reshard_kernel", "algorithmic_bytes_per_launch": alg, "kernel_ms_avg": k_ms},
        "e2e": {"value": moved_all * steps / e2e_ms / 1e6, "unit": UNIT, "ms_per_step": e2e_ms / steps,
                "h2d_bytes_per_step": r["h2d"] / steps, "d2h_bytes_per_step": r["d2h"] / steps},
        "gpu_launches": 2 * steps * world,
        "clocks": r["clocks"],
    }
    nv = r.get("naive")
    if nv and "error" not in nv:
        def nd(key, fused, ms_key):
            ms = min(nv[ms_key])
            b = nv[key]["bytes_read"] + nv[key]["bytes_written"]
            return {"ms": ms, "launches": nv[key]["launches"], "hbm_bytes_by_construction": b,
                    "passes_vs_direct": b / fused["algorithmic_traffic_bytes"], "GBps": b / ms / 1e6,
                    "fused_speedup": ms / fused["kernel_ms_avg"]}
        line["naive_3stage"] = {"what": "PAPER.md Table 1 'Naive' on one device: permute -> exchange (-> scatter) through a staging "
                                        "buffer, plain ld/st kernels, same plan and bit-identical result; context, not the metric",
                                "tp2ep": nd("tp2ep", d_t2e, "tp2ep_ms"), "ep2tp": nd("ep2tp", d_e2t, "ep2tp_ms"),
                                "scratch_GB": nv["tp2ep"]["scratch_bytes"] / 1e9}
        line["gpu_launches"] += 2 * (nv["tp2ep"]["launches"] + nv["ep2tp"]["launches"])
    elif nv:
        line["naive_3stage"] = nv
    pool_bytes = r["pool"]
    del r
    # the other BASELINE.json configs, driver-timed in the same run (1 GPU, default workload only)
    if world == 1 and not args.no_other_configs and args.config == "qwen3_235b" and args.pool == "roomy" \
            and not args.layers and args.n_req < 0 and not args.w_orient and not args.w_inplace:
        torch.cuda.empty_cache()
        others = {}
        for key, name, pool_policy, cap, over in OTHER_CONFIGS:
            try:
                ro = run_moebius(args, env, name, pool_policy, cap, min(steps, 10), 3, full=False, overrides=over)
                others[key] = other_config_entry(ro, peak)
                line["gpu_launches"] += 2 * ro["steps"]
                del ro
            except Exception as e:      # one failing side workload must not cost the headline line
                others[key] = {"error": repr(e)[:300]}
            torch.cuda.empty_cache()
        line["other_configs"] = others
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(cfg, args.cpu_sample_requests, pool_bytes)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
