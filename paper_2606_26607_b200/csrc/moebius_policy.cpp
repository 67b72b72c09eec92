// moebius_policy.cpp -- the switch coordinator's policy (§4.5) and the KV-capacity
// check that precedes every switch.  Host only.
// Product code: shares nothing with oracle/.
#include <algorithm>
#include <cstring>
#include <new>
#include <vector>

#include "moebius_host.h"

using namespace moebius;

struct moebius_policy {
  moebius_policy_config_t cfg;
  int mode;
  std::vector<int64_t> ring;   // the last W counts
  int64_t sum;                 // of the ring
  int64_t seen;                // samples so far
  bool has_event;              // a switch or a cancelled attempt has happened
  double t_last;               // its time
};

extern "C" {

int moebius_policy_preset(int kind, double T_h, double cooldown_s, moebius_policy_config_t* out) {
  if (!out || out->struct_size != sizeof(moebius_policy_config_t)) return MOEBIUS_E_INVAL;
  if (!(T_h >= 0) || !(cooldown_s >= 0)) return MOEBIUS_E_INVAL;
  out->T_h = T_h;
  out->cooldown_s = cooldown_s;
  if (kind == MOEBIUS_POLICY_INTERACTIVE) {        // T_l = 0.8 T_h, W = 8
    out->T_l = 0.8 * T_h;
    out->W = 8;
  } else if (kind == MOEBIUS_POLICY_ROLLOUT) {     // T_l = T_h, W = 1
    out->T_l = T_h;
    out->W = 1;
  } else {
    return MOEBIUS_E_INVAL;
  }
  return MOEBIUS_OK;
}

int moebius_policy_create(const moebius_policy_config_t* c, moebius_mode_t initial_mode, moebius_policy_t** out) {
  if (!c || !out || c->struct_size != sizeof(moebius_policy_config_t)) return MOEBIUS_E_INVAL;
  *out = nullptr;
  if (!(c->T_l <= c->T_h) || c->W < 1 || c->W > (1 << 20) || !(c->cooldown_s >= 0)) return MOEBIUS_E_INVAL;
  if (initial_mode != MOEBIUS_TP && initial_mode != MOEBIUS_EP) return MOEBIUS_E_INVAL;
  moebius_policy* p = new (std::nothrow) moebius_policy();
  if (!p) return MOEBIUS_E_INVAL;
  p->cfg = *c;
  p->mode = initial_mode;
  p->ring.assign((size_t)c->W, 0);
  p->sum = 0;
  p->seen = 0;
  p->has_event = false;
  p->t_last = 0.0;
  *out = p;
  return MOEBIUS_OK;
}

void moebius_policy_destroy(moebius_policy_t* p) { delete p; }

int moebius_policy_mode(const moebius_policy_t* p) { return p ? p->mode : MOEBIUS_E_INVAL; }

// "checks that the target mode has enough KV capacity for the current live requests".
// TP: one shared table, every rank stores its head shard of every request -> all pages in one pool.
// EP: the requests are partitioned first; each rank must hold its own share.
int moebius_capacity_check(moebius_ctx_t* x, moebius_mode_t to, int32_t n_req, const int32_t* seq_lens) {
  if (!x || n_req < 0 || (n_req > 0 && !seq_lens)) return MOEBIUS_E_INVAL;
  if (to != MOEBIUS_TP && to != MOEBIUS_EP) return MOEBIUS_E_INVAL;
  if (n_req > x->cfg.max_requests) return MOEBIUS_E_CAPACITY;
  const int pg = x->cfg.page_tokens, R = x->cfg.R;
  int64_t total = 0;
  for (int i = 0; i < n_req; ++i) {
    if (seq_lens[i] < 0) return MOEBIUS_E_INVAL;
    int64_t np = (seq_lens[i] + pg - 1) / pg;
    if (np > x->cfg.max_pages_per_request) return MOEBIUS_E_CAPACITY;
    total += np;
  }
  if (to == MOEBIUS_TP) return total <= x->pages_tp ? MOEBIUS_OK : MOEBIUS_E_CAPACITY;
  PlanScratch& W = x->scratch;
  W.owner.assign((size_t)n_req, -1);
  lpt_partition(n_req, seq_lens, R, W, W.owner.data());
  W.used.assign((size_t)R, 0);
  for (int i = 0; i < n_req; ++i) {
    int64_t& u = W.used[(size_t)W.owner[(size_t)i]];
    u += (seq_lens[i] + pg - 1) / pg;
    if (u > x->pages_ep) return MOEBIUS_E_CAPACITY;
  }
  return MOEBIUS_OK;
}

// One sample of the control signal, taken after a decode iteration.
int moebius_policy_step(moebius_policy_t* p, moebius_ctx_t* ctx, double now_s, int32_t n_req,
                        const int32_t* seq_lens, int32_t* decision, int32_t* mode_after) {
  if (!p || !decision || n_req < 0) return MOEBIUS_E_INVAL;
  // everything that can be rejected is rejected before the window or the cooldown clock move
  if (ctx && n_req > 0) {
    if (!seq_lens) return MOEBIUS_E_INVAL;
    for (int32_t i = 0; i < n_req; ++i) if (seq_lens[i] < 0) return MOEBIUS_E_INVAL;
  }
  const moebius_policy_config_t& c = p->cfg;
  // the window always advances, cooling down or not (reading P2)
  const size_t slot = (size_t)(p->seen % c.W);
  p->sum += (int64_t)n_req - p->ring[slot];
  p->ring[slot] = n_req;
  p->seen++;
  *decision = MOEBIUS_DECISION_STAY;
  if (mode_after) *mode_after = p->mode;
  if (p->has_event && now_s < p->t_last + c.cooldown_s) return MOEBIUS_OK;
  int want = -1;
  if (p->mode == MOEBIUS_TP) {
    if ((double)n_req > c.T_h) want = MOEBIUS_EP;                       // latest count exceeds T_h
  } else if (p->seen >= c.W) {
    if ((double)p->sum / (double)c.W < c.T_l) want = MOEBIUS_TP;       // mean of the last W below T_l
  }
  if (want < 0) return MOEBIUS_OK;
  if (ctx) {
    int rc = moebius_capacity_check(ctx, (moebius_mode_t)want, n_req, seq_lens);
    if (rc != MOEBIUS_OK && rc != MOEBIUS_E_CAPACITY) return rc;         // a failed call starts no cooldown
    if (rc == MOEBIUS_E_CAPACITY) {                                      // cancel, retry after the cooldown
      p->has_event = true;
      p->t_last = now_s;
      *decision = MOEBIUS_DECISION_CANCELLED;
      return MOEBIUS_OK;
    }
  }
  p->has_event = true;
  p->t_last = now_s;
  p->mode = want;
  *decision = MOEBIUS_DECISION_SWITCH;
  if (mode_after) *mode_after = p->mode;
  return MOEBIUS_OK;
}

// "probes EP and TP decode cost over a small set of batch sizes and chooses the
// crossover as the initial threshold" (reading P4: linear interpolation between the probes).
int moebius_policy_calibrate(int32_t n, const int32_t* batch_sizes, const double* tp_cost, const double* ep_cost,
                             int32_t* T_h_out) {
  if (n < 1 || !batch_sizes || !tp_cost || !ep_cost || !T_h_out) return MOEBIUS_E_INVAL;
  for (int k = 1; k < n; ++k) if (batch_sizes[k] <= batch_sizes[k - 1]) return MOEBIUS_E_INVAL;
  bool tp_always = true;
  for (int k = 0; k < n; ++k) if (!(ep_cost[k] - tp_cost[k] > 0)) tp_always = false;
  if (tp_always) { *T_h_out = batch_sizes[n - 1]; return MOEBIUS_OK; }
  if (!(ep_cost[0] - tp_cost[0] > 0)) { *T_h_out = batch_sizes[0]; return MOEBIUS_OK; }
  for (int k = 1; k < n; ++k) {
    const double d0 = ep_cost[k - 1] - tp_cost[k - 1], d1 = ep_cost[k] - tp_cost[k];
    if (d1 <= 0 && d0 > 0) {
      const double b0 = batch_sizes[k - 1], b1 = batch_sizes[k];
      const double xo = b0 + (b1 - b0) * d0 / (d0 - d1);
      *T_h_out = (int32_t)(xo + 0.5);
      return MOEBIUS_OK;
    }
  }
  *T_h_out = batch_sizes[n - 1];
  return MOEBIUS_OK;
}

}  // extern "C"
