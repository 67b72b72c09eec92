"""Pins for oracle/policy.py (§4.5, values :241).  No GPU.  A hand-worked trace, an
independent brute-force restatement over the whole history, the properties the paper states
(hysteresis, cooldown bounds the switching rate, rollout drains monotonically -> two switches), and
closed forms for the calibration crossover."""
import json
import os

import numpy as np
import pytest

from oracle import policy as P

NAME = {P.STAY: "stay", P.SWITCH: "switch", P.CANCELLED: "cancelled"}
MODE = {P.TP: "TP", P.EP: "EP"}


def test_golden_trace(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "policy_trace.json")))
    i = g["inputs"]
    c = P.Coordinator(P.TP, i["T_h"], i["T_l"], i["W"], i["C"])
    for (t, n, fits), (dec, mode) in zip(g["trace"], g["expected"]):
        d, m = c.step(t, n, lambda _mode, f=fits: f)
        assert (NAME[d], MODE[m]) == (dec, mode), (t, n)


def brute_force(trace, mode, T_h, T_l, W, C, fits):
    """The same policy restated over the full history: at step k look back at everything."""
    out, events = [], []          # events: times of switches / cancelled attempts
    for k, (t, n) in enumerate(trace):
        cooling = any(t < te + C for te in events[-1:])
        dec = P.STAY
        if not cooling:
            if mode == P.TP:
                want = P.EP if n > T_h else None
            else:
                hist = [c for _, c in trace[:k + 1]]
                want = P.TP if len(hist) >= W and np.mean(hist[-W:]) < T_l else None
            if want is not None:
                events.append(t)
                if fits(k, want):
                    mode, dec = want, P.SWITCH
                else:
                    dec = P.CANCELLED
        out.append((dec, mode))
    return out


@pytest.mark.parametrize("seed", range(6))
@pytest.mark.parametrize("kind", ["interactive", "rollout"])
def test_against_brute_force_on_random_traces(kind, seed):
    rng = np.random.default_rng(seed)
    par = P.preset(kind, T_h=32, cooldown_s=0.5)
    n = 400
    t = np.cumsum(rng.uniform(0.01, 0.08, size=n))
    load = np.clip(30 + 25 * np.sin(np.arange(n) / 17.0) + rng.normal(0, 8, n), 0, None).astype(int)
    fit_draw = rng.random(n) > 0.5
    trace = list(zip(t.tolist(), load.tolist()))
    c = P.Coordinator(P.TP, par["T_h"], par["T_l"], par["W"], par["C"])
    got = [c.step(tt, nn, lambda m, k=k: bool(fit_draw[k])) for k, (tt, nn) in enumerate(trace)]
    want = brute_force(trace, P.TP, par["T_h"], par["T_l"], par["W"], par["C"], lambda k, m: bool(fit_draw[k]))
    assert got == want
    assert any(d == P.SWITCH for d, _ in got) and any(d == P.CANCELLED for d, _ in got)


def test_properties_hysteresis_and_cooldown():
    par = P.preset("interactive")          # T_h 256, T_l 204.8, W 8, C 5 s
    assert par == dict(T_h=256.0, T_l=0.8 * 256.0, W=8, C=5.0)
    c = P.Coordinator(P.EP, **{k: par[k] for k in ("T_h", "T_l", "W", "C")})
    # counts that wander inside the band [T_l, T_h] never trigger EP -> TP (hysteresis) ...
    for k in range(200):
        d, m = c.step(0.05 * k, 205 + (k * 7) % 50, lambda m: True)
        assert d == P.STAY and m == P.EP
    # ... and in TP the same counts never trigger TP -> EP
    c = P.Coordinator(P.TP, **{k: par[k] for k in ("T_h", "T_l", "W", "C")})
    for k in range(200):
        assert c.step(0.05 * k, 205 + (k * 7) % 50, lambda m: True) == (P.STAY, P.TP)
    # a single dip does not flip EP (the window mean stays above T_l), a sustained one does
    c = P.Coordinator(P.EP, **{k: par[k] for k in ("T_h", "T_l", "W", "C")})
    seq = [300] * 8 + [0] + [300] * 8 + [100] * 8
    decs = [c.step(0.05 * k, n, lambda m: True)[0] for k, n in enumerate(seq)]
    assert decs[8] == P.STAY and decs.count(P.SWITCH) == 1 and decs.index(P.SWITCH) > 17
    # cooldown bounds the switching rate: alternating extremes switch at most once per C seconds
    c = P.Coordinator(P.TP, T_h=10, T_l=10, W=1, C=5.0)
    times = []
    for k in range(2000):
        d, _ = c.step(0.01 * k, 1000 if (k // 3) % 2 == 0 else 0, lambda m: True)
        if d == P.SWITCH:
            times.append(0.01 * k)
    assert len(times) >= 3 and min(np.diff(times)) >= 5.0 - 1e-9


def test_rollout_burst_then_monotone_drain():
    """rollout 'arrives as one burst and then drains monotonically': with T_l = T_h, W = 1
    the policy enters EP at the burst and returns to TP once, when the count crosses T_h downwards."""
    par = P.preset("rollout")
    c = P.Coordinator(P.TP, par["T_h"], par["T_l"], par["W"], par["C"])
    counts = [0] + [int(2048 * np.exp(-k / 900.0)) for k in range(4000)]
    sw = []
    for k, n in enumerate(counts):
        d, m = c.step(0.03 * k, n, lambda m: True)
        if d == P.SWITCH:
            sw.append((k, m, n))
    assert [m for _, m, _ in sw] == [P.EP, P.TP]
    assert sw[0][0] == 1 and sw[1][2] < 256 and counts[sw[1][0] - 1] >= 256


def test_calibration_crossover():
    b = [8, 32, 128, 512]
    # linear costs crossing at 100: tp = 1 + b/50, ep = 2 + b/100  -> equal at b = 100
    tp = [1 + x / 50 for x in b]
    ep = [2 + x / 100 for x in b]
    assert P.calibrate_crossover(b, tp, ep) == 100
    assert P.calibrate_crossover(b, [1, 1, 1, 1], [2, 2, 2, 2]) == 512      # EP never cheaper
    assert P.calibrate_crossover(b, [2, 2, 2, 2], [1, 1, 1, 1]) == 8        # EP always cheaper
    assert P.calibrate_crossover([10, 20], [1.0, 3.0], [2.0, 2.0]) == 15    # d = +1, -1 -> midpoint
