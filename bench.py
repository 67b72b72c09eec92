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
    ap.add_argument("--kv-rounds", type=int, default=0, help="max dependent KV rounds before chains are cut by staging (tuning)")
    ap.add_argument("--w-orient", type=int, default=0, choices=[0, 1],
                    help="0: gate,up [E,H,I], down [E,I,H] (BASELINE.json, the headline); 1: the paper's W13 [E,2I,H], W2 [E,H,I] (named in config.workload)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
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


def committed_traffic(config_name):
    """DRAM bytes per launch of the reshard kernel from the committed ncu --set full capture
    (profiles/roofline_traffic.json-like text file written by hand from the capture), or None."""
    p = os.path.join(ROOT, "profiles", "traffic_%s.txt" % config_name)
    if not os.path.exists(p):
        return None
    for line in open(p):
        if line.startswith("traffic_bytes_per_launch="):
            return float(line.split("=", 1)[1])
    return None


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

def oracle_sample(cfg, n_sample_req, seed=0):
    """Logical state of the bounded sample: layer 0 of the expert weights (gate, up, down, all E
    experts) and layer 0's K and V of the first `n_sample_req` requests of the workload."""
    rng = np.random.default_rng(seed)
    dt = {"bf16": np.uint16, "fp32": np.float32, "fp8_e4m3_b128": np.uint8}[cfg.w_dtype]
    W = {}
    for kind in cfg.w_kinds:
        shape = wl.weight_shape(cfg, kind)
        if dt == np.float32:
            W[kind] = rng.standard_normal(shape, dtype=np.float32)
        else:   # opaque bit patterns: generation cost is excluded from the timing anyway
            W[kind] = rng.integers(0, np.iinfo(dt).max, size=shape, dtype=dt, endpoint=True)
    lens = wl.draw_seq_lens(cfg)[:n_sample_req]
    KV = [{i: wl.gen_kv_request(cfg, 0, kvi, i, int(n)) for i, n in enumerate(lens)} for kvi in range(2)]
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


def time_oracle(cfg, n_sample_req, steps, warmup, pool_bytes):
    W, lens, KV = oracle_sample(cfg, n_sample_req)
    for _ in range(warmup):
        oracle_round_trip(cfg, W, lens, KV, pool_bytes)
    t0 = time.perf_counter()
    for _ in range(steps):
        owner = oracle_round_trip(cfg, W, lens, KV, pool_bytes)
    dt = time.perf_counter() - t0
    moved = steps * oracle_sample_moved(cfg, lens, owner)
    sample = ("layer 0 of %d: %s of all %d experts + K and V pools of the first %d of %d requests; "
              "one TP->EP->TP round trip per step" % (cfg.L, "/".join(cfg.w_kinds), cfg.E, len(lens), cfg.n_req))
    return {"value": moved / dt / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
            "seconds": dt, "ms_per_step": dt / steps * 1e3}


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
                             "sample": r["sample"]},
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


def run_moebius(args):
    import torch
    import torch.distributed as dist

    import paper_2606_26607_b200 as mb   # fails loudly if libmoebius.so is missing: no CPU fallback

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device; there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    cfg = wl.get_config(args.config)
    if args.layers:
        cfg = cfg.with_(L=args.layers, name="%s[L=%d]" % (cfg.name, args.layers))
    if args.w_orient:
        cfg = cfg.with_(w_orient=1, name="%s[w_orient=1]" % cfg.name)
    lens = wl.draw_seq_lens(cfg)
    pool = wl.kv_pool_bytes(cfg, lens, args.pool)
    if args.n_req >= 0:
        lens = lens[:args.n_req]
        cfg = cfg.with_(n_req=args.n_req, name="%s[n_req=%d]" % (cfg.name, args.n_req))
    mp = int(max([1] + [(int(x) + cfg.page - 1) // cfg.page for x in lens]))
    c = mb.make_config(R=cfg.R, L=cfg.L, E=cfg.E, H=cfg.H, I=cfg.I, w_dtype=cfg.w_dtype, kv_heads=cfg.kv_heads,
                       head_dim=cfg.head_dim, page_tokens=cfg.page, kv_pool_bytes_per_rank_layer=pool,
                       max_requests=max(len(lens), 1), max_pages_per_request=mp, staging_cap_bytes=0,
                       w_orient=cfg.w_orient)
    probe = mb.Session(c)
    resident = probe.layout.resident_bytes
    probe.close()
    c.staging_cap_bytes = int(args.staging_cap_frac * resident)   # BASELINE.json: cap at ~2.4% of resident bytes
    sess = mb.Session(c, device=dev)
    lay = sess.layout
    if args.launch:
        a, b, u = (int(x) for x in args.launch.split(","))
        mb.moebius_set_launch(sess.ctx, a, b, u)
    if args.tma:
        a, b, u = (int(x) for x in args.tma.split(","))
        mb.moebius_set_tma(sess.ctx, a, b, u)
    if args.kv_rounds:
        mb.moebius_set_kv_rounds(sess.ctx, args.kv_rounds)
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
    for w in range(max(args.warmup, 1)):
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
    for _ in range(args.steps):
        sess.reshard(plan_t2e)
        sess.reshard(plan_e2t)
    e1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    dev_ms = e0.elapsed_time(e1)
    if args.profile_region:
        torch.cuda.cudart().cudaProfilerStop()
    hist = mb.moebius_kernel_ms_history(sess.ctx, 64)[-2 * args.steps:]
    k_t2e, k_e2t = hist[0::2], hist[1::2]
    # context: a plain device-to-device copy of a weight slot on this box, now (read + write bytes)
    d2d = None
    if cfg.R > 1:
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
    # e2e: host inputs -> plan -> reshard (uploads) -> device->host read-back of the published tables
    host_tables = torch.empty(lay.table_bytes // 4, dtype=torch.int32, pin_memory=True)
    tbl_n = lay.tbl_bt_off + n * mp
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    owner, bt_cur, mode = None, bt, TP
    h2d = d2h = 0
    plan_ms = []
    for _ in range(args.steps):
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
    return locals()


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


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    r = run_moebius(args)
    import torch
    import torch.distributed as dist
    world, rank, cfg, steps = r["world"], r["rank"], r["cfg"], args.steps
    st_t2e, st_e2t = r["st_t2e"], r["st_e2t"]
    moved_step = st_t2e["w_moved"] + st_t2e["kv_moved"] + st_e2t["w_moved"] + st_e2t["kv_moved"]
    (dev_ms, e2e_ms), (moved_all,) = reduce_over_ranks([r["dev_ms"], r["e2e_s"] * 1e3], [float(moved_step)], world, r["dev"])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    hist = r["hist"]
    m = len(hist) // 2 * 2
    hist = hist[len(hist) - m:]
    k_t2e, k_e2t = hist[0::2], hist[1::2]
    avg = lambda x: float(sum(x) / max(len(x), 1))  # noqa: E731
    med = lambda x: float(sorted(x)[len(x) // 2]) if x else None  # noqa: E731
    peak, peak_src = measured_peak()

    def direction(st, ms_list):
        ms = avg(ms_list)
        traffic = st["w_read"] + st["w_relocated"] + st["kv_read"] + st["kv_relocated"]
        moved = st["w_moved"] + st["kv_moved"]
        return {"kernel_ms_avg": ms, "kernel_ms_min": min(ms_list) if ms_list else None, "kernel_ms_median": med(ms_list),
                "moved_bytes": moved, "algorithmic_traffic_bytes": traffic,
                "effective_GBps": moved / ms / 1e6 if ms else None,
                "traffic_GBps": traffic / ms / 1e6 if ms else None,
                "frac_strict_vs_8TBps": 2 * moved / (ms * 1e-3) / 8e12 if ms else None,
                "frac_traffic_vs_measured": traffic / ms / 1e6 / peak if ms else None,
                "units": st["n_units"], "segments": st["n_segments"], "kv_moves": st["n_kv_moves"],
                "kv_rounds": st["n_kv_rounds"], "kv_staged": st["n_kv_staged"]}

    d_t2e, d_e2t = direction(st_t2e, k_t2e), direction(st_e2t, k_e2t)
    # roofline of the dominant (only) kernel: algorithmic bytes per launch / average launch duration
    alg = (d_t2e["algorithmic_traffic_bytes"] + d_e2t["algorithmic_traffic_bytes"]) / 2
    k_ms = avg(k_t2e + k_e2t)
    achieved = alg / k_ms / 1e6
    lay = r["lay"]
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
                     "traffic": committed_traffic(cfg.name), "peak_source": peak_src,
                     "kernel": "moebius_reshard_kernel", "algorithmic_bytes_per_launch": alg, "kernel_ms_avg": k_ms},
        "e2e": {"value": moved_all * steps / e2e_ms / 1e6, "unit": UNIT, "ms_per_step": e2e_ms / steps,
                "h2d_bytes_per_step": r["h2d"] / steps, "d2h_bytes_per_step": r["d2h"] / steps},
        "gpu_launches": 2 * steps * world,
        "clocks": r["clocks"],
    }
    if not args.no_cpu_baseline:
        cb = time_oracle(cfg, args.cpu_sample_requests, 1, 0, r["pool"])
        line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
