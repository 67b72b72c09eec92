"""Switch policy of the coordinator (§4.5), step by step.  TEST INFRASTRUCTURE ONLY.

"The coordinator samples this count once per decode iteration ... When Moebius runs in TP ... the
coordinator switches to EP as soon as the latest count exceeds a high threshold T_h.  When Moebius
runs in EP ... switches back to TP only when the mean count over the last W iterations falls below a
low threshold T_l.  The band T_l <= T_h provides hysteresis, and a cooldown C after every switch
bounds the maximum switching rate."  (:207)
"Before committing a decision, Moebius checks that the target mode has enough KV capacity for the
current live requests ... If the target mode cannot fit the current request and token set, rank 0
cancels the switch and retries after the cooldown."  (:211-213)
Values the paper prints (:241): T_h = 256, C = 5 s; interactive serving T_l = 0.8 T_h, W = 8;
rollout T_l = T_h, W = 1.

Readings where the paper is silent (P1-P4):
  P1  the window holds the last W samples seen, across switches; an EP->TP decision needs W samples.
  P2  cooldown: no decision is taken while now < t_last + C, where t_last is the time of the last
      switch OR of the last cancelled attempt ("retries after the cooldown"); samples still enter
      the window.  Before the first switch there is no cooldown.
  P3  "exceeds" / "falls below" are strict: count > T_h, mean < T_l.
  P4  calibration crossover = the batch size where the probed EP and TP decode costs cross, linearly
      interpolated between the two neighbouring probes (TP cheaper below, EP cheaper above); EP never
      cheaper -> the largest probe, EP always cheaper -> the smallest.  Rounded to nearest integer.
"""
from __future__ import annotations

TP, EP = 0, 1
STAY, SWITCH, CANCELLED = 0, 1, 2


def preset(kind: str, T_h: float = 256.0, cooldown_s: float = 5.0):
    """PAPER.md:241."""
    if kind == "interactive":
        return dict(T_h=T_h, T_l=0.8 * T_h, W=8, C=cooldown_s)
    if kind == "rollout":
        return dict(T_h=T_h, T_l=T_h, W=1, C=cooldown_s)
    raise ValueError(kind)


class Coordinator:
    def __init__(self, mode: int, T_h: float, T_l: float, W: int, C: float):
        if not (T_l <= T_h) or W < 1 or C < 0:
            raise ValueError("need T_l <= T_h, W >= 1, C >= 0")
        self.mode, self.T_h, self.T_l, self.W, self.C = mode, float(T_h), float(T_l), int(W), float(C)
        self.samples = []          # every count seen, oldest first
        self.t_last = None         # time of the last switch or cancelled attempt

    def step(self, now: float, count: int, fits_target) -> tuple:
        """One sample (after a decode iteration).  `fits_target(mode) -> bool` is the KV-capacity check
        of the mode the policy wants to enter.  Returns (decision, mode after the decision)."""
        self.samples.append(int(count))
        if self.t_last is not None and now < self.t_last + self.C:
            return STAY, self.mode                                  # P2: cooling down
        want = None
        if self.mode == TP:
            if count > self.T_h:                                    # latest count exceeds T_h
                want = EP
        else:
            if len(self.samples) >= self.W:                         # P1
                last = self.samples[-self.W:]
                if sum(last) / self.W < self.T_l:                   # mean over the last W below T_l
                    want = TP
        if want is None:
            return STAY, self.mode
        self.t_last = now
        if not fits_target(want):
            return CANCELLED, self.mode                             # cancel, retry after the cooldown
        self.mode = want
        return SWITCH, self.mode


def calibrate_crossover(batch_sizes, tp_cost, ep_cost) -> int:
    """P4.  batch_sizes ascending; costs = decode cost per iteration at each probed batch size."""
    d = [e - t for t, e in zip(tp_cost, ep_cost)]                   # > 0: TP cheaper
    if all(x > 0 for x in d):
        return int(batch_sizes[-1])
    if d[0] <= 0:
        return int(batch_sizes[0])
    for k in range(1, len(d)):
        if d[k] <= 0 < d[k - 1]:
            b0, b1 = batch_sizes[k - 1], batch_sizes[k]
            x = b0 + (b1 - b0) * d[k - 1] / (d[k - 1] - d[k])
            return int(x + 0.5)
    return int(batch_sizes[-1])
