// moebius_plan.cpp -- host side of the C ABI: region map (§4.2), the weight plan
// (§3.1), request ownership and target block tables (§3.2), the KV
// page-move list with its dependency rounds and bounded staging, and the byte accounting.
// Product code: it shares nothing with oracle/.
#include <algorithm>
#include <functional>
#include <cstdlib>
#include <cstring>
#include <new>
#include <numeric>

#include "moebius_host.h"

using namespace moebius;

namespace {

int64_t align_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }
int dtype_bytes(int d) { return d == MOEBIUS_BF16 ? 2 : d == MOEBIUS_FP32 ? 4 : d == MOEBIUS_FP8_E4M3_B128 ? 1 : 0; }

// 128-wide blocks of the intermediate axis that TP shard r touches (reading A13)
void scale_blocks(int r, int R, int I, int* lo, int* hi) {
  int w = I / R;
  *lo = (r * w) / 128;
  *hi = ((r + 1) * w - 1) / 128 + 1;
}

constexpr int kMaxLevelCap = 1024;   // hard bound on dependency rounds (counters: kMaxCounters)
constexpr int kS2BlocksPerRank = 64;  // S2: an in-place object is cut into about this many blocks per rank

}  // namespace

// Shapes the TMA path can take (see moebius_units.h PATH_TMA).  Box dimensions are limited to 256
// elements (uint32 elements here, so a run of at most 1024 bytes) and a unit must fit one stage.
void moebius::tma_geometry(moebius_ctx* x) {
  const moebius_config_t& c = x->cfg;
  const int64_t run_gu = (int64_t)(c.I / c.R) * x->wb;
  x->xt_ok = c.R > 1 && run_gu <= 1024 && run_gu * c.R <= x->stage_bytes && c.R <= 256;
  x->xt_rows = x->xt_ok ? (int)std::min<int64_t>(256, x->stage_bytes / (run_gu * c.R)) : 0;
  x->kt_ok = x->run_kv <= 1024 && c.page_tokens <= 256 && x->G <= 256 && x->ep_page_bytes <= x->stage_bytes &&
             x->ep_page_bytes % 128 == 0;
  x->kt_pools = x->kt_ok ? (int)std::min<int64_t>(x->stage_bytes / x->ep_page_bytes, 2 * (int64_t)c.L) : 0;
}

extern "C" {

const char* moebius_status_str(int s) {
  switch (s) {
    case MOEBIUS_OK: return "ok";
    case MOEBIUS_E_INVAL: return "invalid argument";
    case MOEBIUS_E_CAPACITY: return "target mode cannot hold the live requests";
    case MOEBIUS_E_STAGING: return "staging buffer too small";
    case MOEBIUS_E_STATE: return "wrong state";
    case MOEBIUS_E_CUDA: return "CUDA error or no device";
  }
  return "unknown";
}

int moebius_version(void) { return 1; }

int moebius_create(const moebius_config_t* c, moebius_ctx_t** out) {
  if (!c || !out || c->struct_size != sizeof(moebius_config_t)) return MOEBIUS_E_INVAL;
  *out = nullptr;
  const int R = c->R, L = c->L, E = c->E, H = c->H, I = c->I;
  if (R < 1 || L < 1 || E < 1 || H < 1 || I < 1 || R > 64) return MOEBIUS_E_INVAL;
  if (E % R || I % R) return MOEBIUS_E_INVAL;
  if (c->w_orient != 0 && c->w_orient != 1) return MOEBIUS_E_INVAL;
  const int wb = dtype_bytes(c->w_dtype);
  const int kvb = (c->kv_dtype == MOEBIUS_BF16 || c->kv_dtype == MOEBIUS_FP32) ? dtype_bytes(c->kv_dtype) : 0;
  if (!wb || !kvb) return MOEBIUS_E_INVAL;
  if (((int64_t)(I / R) * wb) % 16) return MOEBIUS_E_INVAL;  // reading A3
  if (c->w_dtype == MOEBIUS_FP8_E4M3_B128 && (H % 128 || I % 128)) return MOEBIUS_E_INVAL;
  const int Hkv = c->kv_heads, D = c->head_dim, pg = c->page_tokens;
  if (Hkv < 1 || D < 1 || pg < 1 || pg > 255) return MOEBIUS_E_INVAL;
  if (!(Hkv % R == 0 || R % Hkv == 0)) return MOEBIUS_E_INVAL;
  if (c->max_requests < 0 || c->max_pages_per_request < 0) return MOEBIUS_E_INVAL;
  if (c->staging_cap_bytes < 0 || c->kv_pool_bytes_per_rank_layer < 0) return MOEBIUS_E_INVAL;
  if (c->attn_mode < MOEBIUS_ATTN_NONE || c->attn_mode > MOEBIUS_ATTN_GATHER) return MOEBIUS_E_INVAL;
  if (c->attn_mode != MOEBIUS_ATTN_NONE) {
    const int Hq = c->n_q_heads;
    if (Hq < 1 || Hq % R || Hq % Hkv) return MOEBIUS_E_INVAL;
    if (((int64_t)D * H * 2) % 16 || ((int64_t)(Hq / R) * D * 2) % 16) return MOEBIUS_E_INVAL;
  }

  moebius_ctx* x = new (std::nothrow) moebius_ctx();
  if (!x) return MOEBIUS_E_INVAL;
  x->cfg = *c;
  x->wb = wb;
  x->kvb = kvb;
  if (c->w_orient == 0) {   // BASELINE.json: gate, up [E,H,I], down [E,I,H]
    x->n_obj = 3;
    x->obj[0] = {MOEBIUS_T_GATE, MOEBIUS_T_GATE_SCALE, 0, 1, 0, 1};
    x->obj[1] = {MOEBIUS_T_UP, MOEBIUS_T_UP_SCALE, 1, 1, 0, 1};
    x->obj[2] = {MOEBIUS_T_DOWN, MOEBIUS_T_DOWN_SCALE, 2, 1, 1, 1};
  } else {                  // W13 [E,2I,H] (gate rows then up rows), W2 [E,H,I]
    x->n_obj = 2;
    x->obj[0] = {MOEBIUS_T_W13, MOEBIUS_T_W13_SCALE, 0, 2, 1, 2};
    x->obj[1] = {MOEBIUS_T_W2, MOEBIUS_T_W2_SCALE, 2, 1, 0, 1};
    x->obj[2] = {-1, -1, 0, 0, 0, 0};
  }
  x->ep_shift = 0;
  if (R > 1) for (int o = 0; o < x->n_obj; ++o) x->ep_shift = std::max(x->ep_shift, x->obj[o].n_slots);
  x->hpr = Hkv >= R ? Hkv / R : 1;
  x->rep = Hkv >= R ? 1 : R / Hkv;
  x->G = Hkv >= R ? R : Hkv;
  x->run_kv = (int64_t)x->hpr * D * kvb;
  if (x->run_kv % 16) { delete x; return MOEBIUS_E_INVAL; }
  x->tp_page_bytes = (int64_t)pg * x->run_kv;
  x->ep_page_bytes = x->tp_page_bytes * x->G;
  x->pool_bytes = c->kv_pool_bytes_per_rank_layer;
  if (x->pool_bytes % x->ep_page_bytes || x->ep_page_bytes > (1 << 30)) { delete x; return MOEBIUS_E_INVAL; }
  int64_t pe = x->pool_bytes / x->ep_page_bytes;
  if (pe * x->G > INT32_MAX) { delete x; return MOEBIUS_E_INVAL; }
  x->pages_ep = (int32_t)pe;
  x->pages_tp = (int32_t)(pe * x->G);

  // rank region: [weight chain: 3L+ep_shift slots][TP scales][EP scales][2L KV pools]
  x->S = align_up((int64_t)(E / R) * H * I * wb, 256);
  x->w_off = 0;
  // How far the EP view of an object sits behind its TP view.  The largest object's size makes every
  // move out of place (S1; PAPER.md:150-156 at object grain).  When the cap does not allow that many
  // spare slots the shift shrinks -- to 0 if need be, where both views alias the same bytes -- and the
  // objects that overlap themselves take the in-place path (S2, s2_object below), with at least a fifth of
  // the cap kept for staging.
  if (R > 1) {
    const int max_obj = x->ep_shift;
    int64_t dup = 0;
    if (c->attn_mode == MOEBIUS_ATTN_DUAL)
      dup = (2 * (int64_t)(c->n_q_heads / R) + 2 * (int64_t)x->hpr) * D * H * 2 * L * R;
    int sft = max_obj;
    if (c->w_inplace) sft = 0;
    else if (c->staging_cap_bytes > 0)
      while (sft > 0 && (int64_t)sft * x->S * R + dup > (sft == max_obj ? c->staging_cap_bytes : c->staging_cap_bytes / 5 * 4)) --sft;
    x->ep_shift = sft;
  }
  int64_t off = (int64_t)(3 * L + x->ep_shift) * x->S;
  x->scale_tp_layer = x->scale_ep_layer = 0;
  memset(x->sg, 0, sizeof(x->sg));
  if (c->w_dtype == MOEBIUS_FP8_E4M3_B128) {
    int nb_max = 0;
    for (int r = 0; r < R; ++r) { int lo, hi; scale_blocks(r, R, I, &lo, &hi); nb_max = std::max(nb_max, hi - lo); }
    for (int m = 0; m < x->n_obj; ++m) {
      const int mult = x->obj[m].row_mult;
      x->sg[m].tp_bytes = align_up((int64_t)E * (H / 128) * nb_max * mult * 4, 256);
      x->sg[m].ep_bytes = align_up((int64_t)(E / R) * (H / 128) * (I / 128) * mult * 4, 256);
      x->scale_tp_layer += x->sg[m].tp_bytes;
      x->scale_ep_layer += x->sg[m].ep_bytes;
    }
  }
  x->scale_tp_off = off;  off += x->scale_tp_layer * L;
  x->scale_ep_off = off;  off += x->scale_ep_layer * L;
  // attention projections, bf16: wq [Hq,D,H], wk/wv [Hkv,D,H], wo [H,Hq,D] (reading A19)
  x->attn_off = align_up(off, 256);
  x->attn_layer_bytes = x->attn_full_bytes = x->attn_dup_bytes = 0;
  memset(x->attn_full_off, 0, sizeof(x->attn_full_off)); memset(x->attn_shard_off, 0, sizeof(x->attn_shard_off));
  memset(x->attn_full_sz, 0, sizeof(x->attn_full_sz));   memset(x->attn_shard_sz, 0, sizeof(x->attn_shard_sz));
  if (c->attn_mode != MOEBIUS_ATTN_NONE) {
    const int64_t head = (int64_t)D * H * 2;
    const int Hq = c->n_q_heads;
    const int64_t full[4] = {Hq * head, Hkv * head, Hkv * head, Hq * head};
    const int64_t shard[4] = {(Hq / R) * head, x->hpr * head, x->hpr * head, (Hq / R) * head};
    int64_t at = 0, sum_full = 0, sum_shard = 0;
    for (int t = 0; t < 4; ++t) { x->attn_full_off[t] = at; x->attn_full_sz[t] = full[t]; at += align_up(full[t], 256); sum_full += full[t]; }
    for (int t = 0; t < 4; ++t) {
      x->attn_shard_sz[t] = shard[t];
      sum_shard += shard[t];
      if (c->attn_mode == MOEBIUS_ATTN_DUAL) { x->attn_shard_off[t] = at; at += align_up(shard[t], 256); }
    }
    x->attn_layer_bytes = at;
    x->attn_full_bytes = sum_full * L * R;
    x->attn_dup_bytes = c->attn_mode == MOEBIUS_ATTN_DUAL ? sum_shard * L * R : 0;
    off = x->attn_off + x->attn_layer_bytes * L;
  }
  off = align_up(off, 4096);
  x->kv_off = off;        off += 2 * (int64_t)L * x->pool_bytes;
  // the rank's flag page for the device-side round barrier (moebius_reshard_shares): inside the unified
  // buffer, so that a peer GPU reaches it through the same mapping as the data
  off = align_up(off, 4096);
  x->flag_off = off;      off += 4 * (int64_t)kMaxCounters;
  x->rank_stride = align_up(off, 2 << 20);   // 2 MiB: a rank region can be its own physical allocation (moebius_arena_*)

  x->spare_bytes = (int64_t)x->ep_shift * x->S * R;
  x->resident_bytes = (int64_t)3 * L * x->S * R + 2 * (int64_t)L * x->pool_bytes * R + x->attn_full_bytes;
  const int64_t kv_total = 2 * (int64_t)L * x->pool_bytes * R;
  // what dual residency costs beyond the single resident copy: the spare weight slot(s) and, with
  // MOEBIUS_ATTN_DUAL, the duplicated head shards (1.1 GB + 1.7 GB = 2.4 % per GPU)
  const int64_t overhead = x->spare_bytes + x->attn_dup_bytes;
  if (c->staging_cap_bytes == 0) {
    // no bound given: 2% of the KV capacity, and never less than 64 EP pages of every pool (a tiny
    // pool would otherwise get a staging buffer smaller than one page)
    x->staging_bytes = std::max(kv_total / 50, std::min(kv_total, 64 * x->ep_page_bytes * 2 * (int64_t)L));
  } else {
    if (c->staging_cap_bytes < overhead) { delete x; return MOEBIUS_E_STAGING; }
    x->staging_bytes = std::min(c->staging_cap_bytes - overhead, kv_total);
  }
  x->staging_bytes = x->staging_bytes / x->ep_page_bytes * x->ep_page_bytes;
  // S2: the tail half of the staging buffer parks weight blocks, the head stays with the KV schedule
  x->w_stg_bytes = 0;
  x->max_wblk = R > 1 ? (int64_t)L * x->n_obj * 2 * R : 0;     // banded chain: 4 segments of R/2 blocks per link
  if (R > 1) {
    bool s2 = false;
    for (int o = 0; o < x->n_obj; ++o) s2 |= x->obj[o].n_slots > x->ep_shift;
    if (s2) {
      if (c->staging_cap_bytes == 0) {   // no bound given: room to park 2R+2 of the largest EP rows (one expert matrix)
        const int64_t need = (2 * (int64_t)R + 2) * I * H * wb * 2;
        x->staging_bytes = std::max(x->staging_bytes, align_up(2 * need, x->ep_page_bytes));
      }
      x->w_stg_bytes = x->staging_bytes / 2 / 256 * 256;
      x->max_wblk += (int64_t)L * x->n_obj * R * 4 * kS2BlocksPerRank;
    }
  }

  // descriptor buffer: header, counters, segments, KV moves (each live page at most twice), scale copies
  int64_t live_max = std::max<int64_t>((int64_t)x->pages_tp, (int64_t)x->pages_ep * R);
  live_max = std::min<int64_t>(live_max, (int64_t)c->max_requests * c->max_pages_per_request);
  x->max_kv_desc = live_max;
  x->max_c2d = c->w_dtype == MOEBIUS_FP8_E4M3_B128 ? (int64_t)x->n_obj * L * R * R : 0;
  x->max_bulk = c->attn_mode == MOEBIUS_ATTN_GATHER ? (int64_t)L * R * (2 * (int64_t)R + 2 * (int64_t)std::max(R, Hkv)) : 0;
  x->desc_bytes = align_up(kSegOff + (int64_t)(1 + kMaxCounters) * sizeof(PlanHdr) + 2 * (int64_t)kMaxSegs * sizeof(Seg) + x->max_kv_desc * sizeof(KvDesc) +
                               x->max_c2d * sizeof(C2dDesc) + (x->max_bulk + x->max_wblk) * sizeof(BulkDesc) + x->max_wblk * sizeof(WBlk) + 1024, 4096);
  x->table_bytes = align_up(4 * ((int64_t)kTblHdrInts + 2 * (int64_t)c->max_requests +
                                 (int64_t)c->max_requests * c->max_pages_per_request), 256);
  x->bound = false;
  x->base = x->stg = x->desc = nullptr;
  x->tables = nullptr;
  x->active_mode = -1;
  x->switch_count = 0;
  x->ctas_per_sm = 0;
  x->threads = 0;
  x->unit_kb = 0;
  x->kv_max_level = 64;
  x->kv_slice_floor = 0;
  x->chain_bands = 0;
  x->xt_mode = 1;
  x->xt_promo = 0;
  x->use_tma = 1;
  x->n_pipes = 2;
  x->stage_bytes = 48 * 1024;
  // A KV unit is a whole number of EP pages: size the stage to a multiple of the page so that no part of
  // it stays empty, and use the shared memory that frees for more pipes (bytes in flight per SM are
  // what sets the rate: 2 pipes x 2 stages x 48 KB at 16-KB pages; 3 x 2 x 32 KB at 32-KB pages).
  if (x->ep_page_bytes % 128 == 0 && x->ep_page_bytes <= 96 * 1024) {
    const int64_t k = std::max<int64_t>(1, (48 * 1024) / x->ep_page_bytes);
    const int64_t sb = k * x->ep_page_bytes;
    if (sb >= 24 * 1024) {
      x->stage_bytes = sb;
      x->n_pipes = (int)std::max<int64_t>(1, std::min<int64_t>(4, (208 * 1024) / (2 * sb)));
    }
  }
  x->ring_bytes = 2 * x->stage_bytes;
  x->ld_max = 2;
  x->l2_ld = 2;   // loads evict_last, stores unhinted: measured 0.6-1.0 % faster than no hint at every BASELINE shape
  x->l2_st = 0;
  x->def_pipes = x->n_pipes;
  x->def_stage_bytes = x->stage_bytes;
  x->tmaps_valid = false;
  x->prepared = false;
  x->smem_set = 0;
  tma_geometry(x);
  x->n_sm = 0;
  x->timing = 0;
  memset(x->ev, 0, sizeof(x->ev));
  x->ev_count = 0;
  x->ev_valid = false;
  x->has_device = -1;
  x->mailbox = nullptr;
  *out = x;
  return MOEBIUS_OK;
}

void moebius_destroy(moebius_ctx_t* ctx) {
  if (!ctx) return;
  cuda_ctx_destroy(ctx);
  delete ctx;
}

int moebius_layout(const moebius_ctx_t* x, moebius_layout_t* o) {
  if (!x || !o || o->struct_size != sizeof(moebius_layout_t)) return MOEBIUS_E_INVAL;
  o->pages_tp = x->pages_tp;
  o->pages_ep = x->pages_ep;
  o->tp_page_bytes = (int32_t)x->tp_page_bytes;
  o->ep_page_bytes = (int32_t)x->ep_page_bytes;
  o->base_bytes = x->rank_stride * x->cfg.R;
  o->rank_stride_bytes = x->rank_stride;
  o->weight_slot_bytes = x->S;
  o->weight_spare_bytes = x->spare_bytes;
  o->staging_bytes = x->staging_bytes;
  o->desc_bytes = x->desc_bytes;
  o->table_bytes = x->table_bytes;
  o->resident_bytes = x->resident_bytes;
  o->tbl_owner_off = kTblHdrInts;
  o->tbl_lens_off = kTblHdrInts + x->cfg.max_requests;
  o->tbl_bt_off = kTblHdrInts + 2 * x->cfg.max_requests;
  o->tbl_reserved = 0;
  o->attn_full_bytes = x->attn_full_bytes;
  o->attn_dup_bytes = x->attn_dup_bytes;
  o->w_staging_bytes = x->w_stg_bytes;
  o->w_shift_slots = x->ep_shift;
  o->reserved1 = 0;
  return MOEBIUS_OK;
}

int moebius_view(const moebius_ctx_t* x, moebius_mode_t mode, int rank, int layer, int t, moebius_view_t* o) {
  if (!x || !o || o->struct_size != sizeof(moebius_view_t)) return MOEBIUS_E_INVAL;
  const moebius_config_t& c = x->cfg;
  if (rank < 0 || rank >= c.R || layer < 0 || layer >= c.L) return MOEBIUS_E_INVAL;
  if (mode != MOEBIUS_TP && mode != MOEBIUS_EP) return MOEBIUS_E_INVAL;
  const bool tp = mode == MOEBIUS_TP;
  const int64_t rbase = (int64_t)rank * x->rank_stride;
  const int R = c.R, E = c.E, H = c.H, I = c.I;
  for (int i = 0; i < 4; ++i) o->shape[i] = 1;
  int wo = -1, so = -1;   // object whose weight / scale tensor this id names
  for (int o = 0; o < x->n_obj; ++o) {
    if (x->obj[o].tensor_id == t) wo = o;
    if (x->obj[o].scale_id == t) so = o;
  }
  if (wo >= 0) {
    const WObj& ob = x->obj[wo];
    o->offset = rbase + x->w_off + (int64_t)(3 * layer + ob.slot + (tp ? 0 : x->ep_shift)) * x->S;
    o->elem_bytes = x->wb;
    o->ndim = 3;
    o->shape[0] = tp ? E : E / R;
    const int64_t i_dim = (int64_t)(tp ? I / R : I) * ob.row_mult;
    if (!ob.long_run) { o->shape[1] = H; o->shape[2] = i_dim; }   // gate, up, W2: [., H, I]
    else              { o->shape[1] = i_dim; o->shape[2] = H; }   // down, W13:    [., I or 2I, H]
  } else if (t == MOEBIUS_T_KPOOL || t == MOEBIUS_T_VPOOL) {
    int z = 2 * layer + (t - MOEBIUS_T_KPOOL);
    o->offset = rbase + x->kv_off + (int64_t)z * x->pool_bytes;
    o->elem_bytes = x->kvb;
    o->ndim = 4;
    o->shape[0] = tp ? x->pages_tp : x->pages_ep;
    o->shape[1] = c.page_tokens;
    o->shape[2] = tp ? x->hpr : c.kv_heads;
    o->shape[3] = c.head_dim;
  } else if (t >= MOEBIUS_T_WQ && t <= MOEBIUS_T_WO) {
    // PAPER.md:112.  EP: the full projection on every rank.  TP: the rank's head shard -- a dense tensor
    // of its own (MOEBIUS_ATTN_DUAL) or in place inside the full one (MOEBIUS_ATTN_GATHER).
    if (c.attn_mode == MOEBIUS_ATTN_NONE) return MOEBIUS_E_INVAL;
    const int a = t - MOEBIUS_T_WQ, Hq = c.n_q_heads, D = c.head_dim;
    const bool kv = a == 1 || a == 2;
    const int64_t n_full = kv ? c.kv_heads : Hq, n_sh = kv ? x->hpr : Hq / R;
    const int64_t first = kv ? (c.kv_heads >= R ? (int64_t)rank * x->hpr : rank / x->rep) : (int64_t)rank * (Hq / R);
    const int64_t lbase = rbase + x->attn_off + (int64_t)layer * x->attn_layer_bytes;
    o->elem_bytes = 2;
    o->ndim = 3;
    const int64_t heads = tp ? n_sh : n_full;
    if (a != 3) { o->shape[0] = heads; o->shape[1] = D; o->shape[2] = H; }
    else        { o->shape[0] = H; o->shape[1] = heads; o->shape[2] = D; }
    if (!tp) o->offset = lbase + x->attn_full_off[a];
    else if (c.attn_mode == MOEBIUS_ATTN_DUAL) o->offset = lbase + x->attn_shard_off[a];
    else {   // in place: heads [first, first + n_sh) of the full tensor
      o->offset = lbase + x->attn_full_off[a] + first * (a != 3 ? (int64_t)D * H * 2 : (int64_t)D * 2);
      if (a == 3) {
        o->stride[0] = (int64_t)Hq * D; o->stride[1] = D; o->stride[2] = 1; o->stride[3] = 0;
        return MOEBIUS_OK;
      }
    }
  } else if (so >= 0) {
    if (c.w_dtype != MOEBIUS_FP8_E4M3_B128) return MOEBIUS_E_INVAL;
    const WObj& ob = x->obj[so];
    int64_t within = 0;
    for (int mm = 0; mm < so; ++mm) within += tp ? x->sg[mm].tp_bytes : x->sg[mm].ep_bytes;
    o->offset = rbase + (tp ? x->scale_tp_off + layer * x->scale_tp_layer
                            : x->scale_ep_off + layer * x->scale_ep_layer) + within;
    o->elem_bytes = 4;
    o->ndim = 3;
    int lo, hi;
    scale_blocks(rank, R, I, &lo, &hi);
    const int64_t i_dim = (int64_t)(tp ? hi - lo : I / 128) * ob.row_mult;
    o->shape[0] = tp ? E : E / R;
    if (!ob.long_run) { o->shape[1] = H / 128; o->shape[2] = i_dim; }
    else              { o->shape[1] = i_dim; o->shape[2] = H / 128; }
  } else {
    return MOEBIUS_E_INVAL;
  }
  int64_t st = 1;
  for (int i = 3; i >= 0; --i) {
    if (i >= o->ndim) { o->stride[i] = 0; continue; }
    o->stride[i] = st;
    st *= o->shape[i];
  }
  return MOEBIUS_OK;
}

int moebius_active_mode(const moebius_ctx_t* x) { return x ? x->active_mode : MOEBIUS_E_INVAL; }

int moebius_set_tma(moebius_ctx_t* x, int enable, int pipes, int stage_kb) {
  if (!x) return MOEBIUS_E_INVAL;
  if (pipes < 0 || pipes > 8 || stage_kb < 0) return MOEBIUS_E_INVAL;
  int np = pipes > 0 ? pipes : x->def_pipes;
  int64_t sb = stage_kb > 0 ? (int64_t)stage_kb * 1024 : x->def_stage_bytes;
  if ((int64_t)np * 2 * sb > 208 * 1024) return MOEBIUS_E_INVAL;   // 227 KB per CTA minus barriers and slack
  x->use_tma = enable ? 1 : 0;
  x->n_pipes = np;
  x->stage_bytes = sb;
  x->ring_bytes = 2 * sb;
  x->tmaps_valid = false;
  tma_geometry(x);
  return device_prepare(x);   // a bound context re-encodes its tensor maps and shared-memory size here
}

int moebius_set_ring(moebius_ctx_t* x, int ring_kb, int max_loads) {
  if (!x || ring_kb < 0 || max_loads < 0 || max_loads > 7) return MOEBIUS_E_INVAL;
  const int64_t rb = ring_kb > 0 ? (int64_t)ring_kb * 1024 : 2 * x->stage_bytes;
  if (rb < x->stage_bytes || (int64_t)x->n_pipes * rb > 208 * 1024) return MOEBIUS_E_INVAL;
  x->ring_bytes = rb;
  x->ld_max = max_loads > 0 ? max_loads : 2;
  return device_prepare(x);   // the kernel's shared-memory size follows the ring
}

int moebius_set_kv_rounds(moebius_ctx_t* x, int max_level) {
  if (!x || max_level < 0 || max_level > kMaxLevelCap) return MOEBIUS_E_INVAL;
  x->kv_max_level = max_level > 0 ? max_level : 64;
  return MOEBIUS_OK;
}

int moebius_set_xt_mode(moebius_ctx_t* x, int mode) {
  if (!x || mode < 0 || (mode & 15) > 1 || (mode >> 4) > 3) return MOEBIUS_E_INVAL;
  const bool re_encode = (mode >> 4) != x->xt_promo;
  x->xt_mode = mode & 15;
  x->xt_promo = mode >> 4;
  if (re_encode) { x->tmaps_valid = false; return device_prepare(x); }
  return MOEBIUS_OK;
}

int moebius_set_l2_policy(moebius_ctx_t* x, int load_policy, int store_policy) {
  if (!x || load_policy < 0 || load_policy > 4 || store_policy < 0 || store_policy > 4) return MOEBIUS_E_INVAL;
  x->l2_ld = load_policy;
  x->l2_st = store_policy;
  return MOEBIUS_OK;
}

int moebius_set_chain_bands(moebius_ctx_t* x, int enable) {
  if (!x) return MOEBIUS_E_INVAL;
  x->chain_bands = enable ? 1 : 0;
  return MOEBIUS_OK;
}

int moebius_set_kv_slice(moebius_ctx_t* x, int min_units) {
  if (!x || min_units < 0) return MOEBIUS_E_INVAL;
  x->kv_slice_floor = min_units;
  return MOEBIUS_OK;
}

int moebius_set_launch(moebius_ctx_t* x, int ctas_per_sm, int threads, int unit_kb) {
  if (!x) return MOEBIUS_E_INVAL;
  if (threads > 0 && (threads % 32 || threads > 256)) return MOEBIUS_E_INVAL;
  x->ctas_per_sm = ctas_per_sm > 0 ? ctas_per_sm : 0;
  x->threads = threads > 0 ? threads : 0;
  x->unit_kb = unit_kb > 0 ? unit_kb : 0;
  return MOEBIUS_OK;
}

void moebius_plan_destroy(moebius_plan_t* p) {
  if (!p) return;
  image_release(p->ctx, p->buf);
  delete p;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
namespace {

// Split `run` into equal chunks of at most `limit` bytes, each a multiple of 16.
uint32_t pick_chunk(int64_t run, int64_t limit) {
  if (run <= limit) return (uint32_t)run;
  for (int64_t n = (run + limit - 1) / limit; n <= run / 16; ++n)
    if (run % n == 0 && (run / n) % 16 == 0) return (uint32_t)(run / n);
  return 16;
}

struct Chain {
  std::vector<Seg> segs;
  int64_t units = 0;
};

void push_seg(Chain& ch, const Seg& s) {
  if (s.n_units == 0) return;
  ch.segs.push_back(s);
  ch.units += s.n_units;
}

Seg blank_seg() {
  Seg s;
  memset(&s, 0, sizeof(s));
  s.wait_ctr = -1;
  s.signal_ctr = -1;
  s.rep = 1;
  s.chunks_per_run = 1;
  s.rows_per_unit = 1;
  s.groups_per_unit = 1;
  s.pools_per_unit = 1;
  s.row_blocks = 1;
  return s;
}

}  // namespace

// decreasing length, greedy least-loaded rank, deterministic.  Reading A9: ties by
// request id; least loaded = smallest (tokens, requests, rank).
void moebius::lpt_partition(int n_req, const int32_t* seq_lens, int R, PlanScratch& W, int32_t* owner) {
  std::vector<int32_t>& order = W.order;
  order.resize(n_req);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return seq_lens[a] > seq_lens[b]; });
  W.tok.assign(R, 0); W.cnt.assign(R, 0);
  std::vector<int64_t>&tok = W.tok, &cnt = W.cnt;
  for (int i : order) {
    int best = 0;
    for (int r = 1; r < R; ++r)
      if (tok[r] < tok[best] || (tok[r] == tok[best] && cnt[r] < cnt[best])) best = r;
    owner[i] = best;
    tok[best] += seq_lens[i];
    cnt[best] += 1;
  }
}

namespace {

// One moebius_plan call, stage by stage.  The members are what the stages share; every stage returns a
// moebius_status_t and leaves the context untouched on failure (cancel and retry).
struct PlanBuilder {
  moebius_ctx* x;
  const moebius_config_t& c;
  const moebius_mode_t from, to;
  const int32_t n_req;
  const int32_t *seq_lens, *src_owner, *src_bt;
  const int R, L, pg, MP;
  const bool e2t;
  const int n_pools_all;
  const int64_t unit_bytes;
  const int kappa;                       // TP-page granules per EP page
  PlanScratch& W;                        // warm workspace: no fresh multi-megabyte allocation per switch
  std::vector<int32_t>&npages, &owner, &bt;
  std::vector<Move>& mv;
  int64_t total_pages = 0;
  int nm = 0, n_staged = 0, K = 0, pools_per_group = 0, n_pool_groups = 0;
  moebius_plan_t* P = nullptr;
  uint32_t next_ctr = 0;
  uint64_t ub = 0;                       // units of the merged list
  Chain cw, ck, cs, ca;                  // weight chain, KV rounds, scale copies, attention gathers

  PlanBuilder(moebius_ctx* x_, moebius_mode_t from_, moebius_mode_t to_, int32_t n, const int32_t* lens,
              const int32_t* so, const int32_t* sbt)
      : x(x_), c(x_->cfg), from(from_), to(to_), n_req(n), seq_lens(lens), src_owner(so), src_bt(sbt),
        R(c.R), L(c.L), pg(c.page_tokens), MP(c.max_pages_per_request), e2t(from_ == MOEBIUS_EP),
        n_pools_all(2 * c.L), unit_bytes((int64_t)(x_->unit_kb > 0 ? x_->unit_kb : 32) * 1024), kappa(x_->G),
        W(x_->scratch), npages(W.npages), owner(W.owner), bt(W.bt), mv(W.mv) {}

  int fail(int code) { moebius_plan_destroy(P); P = nullptr; return code; }

  // ownership and block tables under the target mode
  int request_state() {
    // ---- request state under the target mode ----------------------------------------------------
    npages.assign(n_req, 0);
    total_pages = 0;
    for (int i = 0; i < n_req; ++i) {
      if (seq_lens[i] < 0) return MOEBIUS_E_INVAL;
      npages[i] = (seq_lens[i] + pg - 1) / pg;
      if (npages[i] > MP) return MOEBIUS_E_INVAL;
      total_pages += npages[i];
      if (e2t && (src_owner[i] < 0 || src_owner[i] >= R)) return MOEBIUS_E_INVAL;
    }
    owner.assign(n_req, -1);
    if (!e2t) {
      lpt_partition(n_req, seq_lens, R, W, owner.data());
    }
    // reading A7: ascending request id, consecutive pages; TP bumps up from 0, EP down from the top.
    // Only the first npages[i] entries of a row are written here; the -1 padding is laid down when
    // the table image is built.
    if (bt.size() < (size_t)n_req * MP) bt.resize((size_t)n_req * MP);
    if (e2t) {
      if (total_pages > x->pages_tp) return MOEBIUS_E_CAPACITY;
      int32_t nxt = 0;
      for (int i = 0; i < n_req; ++i)
        for (int b = 0; b < npages[i]; ++b) bt[(size_t)i * MP + b] = nxt++;
    } else {
      W.used.assign(R, 0);
      std::vector<int64_t>& used = W.used;
      for (int i = 0; i < n_req; ++i) {
        int r = owner[i];
        if (used[r] + npages[i] > x->pages_ep) return MOEBIUS_E_CAPACITY;
        for (int b = 0; b < npages[i]; ++b) bt[(size_t)i * MP + b] = (int32_t)(x->pages_ep - 1 - (used[r] + b));
        used[r] += npages[i];
      }
    }
    return MOEBIUS_OK;
  }

  // one move per live (request, block)
  int kv_moves() {
    // ---- KV page moves (one per live (request, block); layer- and K/V-agnostic) ----
    mv.clear();
    mv.reserve((size_t)total_pages);
    for (int i = 0; i < n_req; ++i) {
      for (int b = 0; b < npages[i]; ++b) {
        Move m;
        m.req = i; m.blk = b;
        int32_t sp = src_bt[(size_t)i * MP + b];
        int32_t dp = bt[(size_t)i * MP + b];
        if (sp < 0 || sp >= (e2t ? x->pages_ep : x->pages_tp)) return MOEBIUS_E_INVAL;
        m.ep_rank = e2t ? src_owner[i] : owner[i];
        m.ep_page = e2t ? sp : dp;
        m.tp_page = e2t ? dp : sp;
        m.ntok = std::min(pg, seq_lens[i] - b * pg);
        m.level = 0; m.slot = -1; m.staged = 0;
        mv.push_back(m);
      }
    }
    nm = (int)mv.size();
    {  // source pages must be unique (per owner under EP, globally under TP)
      std::vector<uint8_t>& seen = W.seen;
      seen.assign((size_t)(e2t ? R : 1) * (e2t ? x->pages_ep : x->pages_tp), 0);
      for (const Move& m : mv) {
        size_t id = e2t ? (size_t)m.ep_rank * x->pages_ep + m.ep_page : (size_t)m.tp_page;
        if (seen[id]) return MOEBIUS_E_INVAL;
        seen[id] = 1;
      }
    }
    return MOEBIUS_OK;
  }

  // hazard graph over the page moves -> dependency rounds + staged pages (bounded staging)
  int kv_schedule() {
    // reader[rank*pages_tp + granule] = move that reads it (TP-page-sized granules of a pool).
    // Hazard graph in CSR form: blk[blk_off[m] .. blk_off[m+1]) = moves that READ what m overwrites
    // (m must run after them); dep[...] is the transpose (who waits for b).
    n_staged = 0; K = 0;
    // Fast path: with the two-ended allocation (reading A7) the targets are TP pages [0, total_pages)
    // on every rank resp. the top used[r] EP pages of rank r.  If every source page lies outside those
    // ranges nothing overwrites a live source: one round, no graph needed.
    bool disjoint = nm > 0;
    if (nm > 0) {
      if (e2t) {
        int64_t min_src = INT64_MAX;
        for (const Move& m : mv) min_src = std::min<int64_t>(min_src, (int64_t)m.ep_page * kappa);
        disjoint = min_src >= total_pages;
      } else {
        int64_t max_src = -1, min_dst = INT64_MAX;
        for (const Move& m : mv) max_src = std::max<int64_t>(max_src, m.tp_page);
        for (int r = 0; r < R; ++r) min_dst = std::min<int64_t>(min_dst, ((int64_t)x->pages_ep - W.used[r]) * kappa);
        disjoint = max_src < min_dst;
      }
    }
    if (nm > 0 && !disjoint) {
      std::vector<int32_t>& reader = W.reader;
      reader.assign((size_t)R * x->pages_tp, -1);
      auto gid = [&](int rank, int64_t gran) { return (size_t)rank * x->pages_tp + (size_t)gran; };
      for (int m = 0; m < nm; ++m) {
        if (e2t) {
          for (int g = 0; g < kappa; ++g) {
            int32_t& rd = reader[gid(mv[m].ep_rank, (int64_t)mv[m].ep_page * kappa + g)];
            if (rd >= 0) return MOEBIUS_E_INVAL;  // source page listed twice
            rd = m;
          }
        } else {
          for (int g = 0; g < x->G; ++g) {
            int32_t& rd = reader[gid((int)tp_src_rank((uint32_t)g, (uint32_t)x->rep, mv[m].ep_rank), mv[m].tp_page)];
            if (rd >= 0) return MOEBIUS_E_INVAL;
            rd = m;
          }
        }
      }
      std::vector<int32_t>&blk_off = W.blk_off, &blk = W.blk, &dep_off = W.dep_off, &dep = W.dep;
      blk_off.assign(nm + 1, 0);
      blk.clear();
      dep_off.assign(nm + 1, 0);
      for (int m = 0; m < nm; ++m) {
        int32_t bl[64];            // R <= 64, kappa <= R
        int nb = 0;
        auto note = [&](int32_t b) {
          if (b < 0) return;
          if (b == m) { mv[m].staged = 1; return; }  // a move whose target overlaps its own source
          bl[nb++] = b;
        };
        if (e2t) for (int j = 0; j < R; ++j) note(reader[gid(j, mv[m].tp_page)]);
        else     for (int g = 0; g < kappa; ++g) note(reader[gid(mv[m].ep_rank, (int64_t)mv[m].ep_page * kappa + g)]);
        if (nb > 1) {
          std::sort(bl, bl + nb);
          nb = (int)(std::unique(bl, bl + nb) - bl);
        }
        for (int i = 0; i < nb; ++i) { blk.push_back(bl[i]); dep_off[bl[i] + 1]++; }
        blk_off[m + 1] = (int32_t)blk.size();
      }
      const bool any_edge = !blk.empty();
      bool any_self = false;
      for (int m = 0; m < nm; ++m) any_self |= mv[m].staged != 0;
      if (any_edge) {
        for (int m = 0; m < nm; ++m) dep_off[m + 1] += dep_off[m];
        dep.resize(blk.size());
        W.dep_cur.assign(dep_off.begin(), dep_off.end() - 1);
        for (int m = 0; m < nm; ++m)
          for (int32_t e = blk_off[m]; e < blk_off[m + 1]; ++e) dep[W.dep_cur[blk[e]]++] = m;
      }
      // Level the DAG of direct moves (Kahn order); a staged move is read in round 0 and written in the
      // last round.  Cycles are broken by staging one move on the cycle.  Chains longer than
      // kv_max_level rounds are CUT rather than staged whole: a move whose level would exceed the
      // limit is staged, so its source is saved in round 0 and everything behind it restarts at
      // level 1.  A round costs a device-wide drain, a staged page one extra copy: short schedules
      // with a few percent of staged pages are the cheapest.
      // No edge at all (the common case: two-ended allocation in a roomy pool) => one round, done.
      if (any_edge) {
        std::vector<uint8_t>&self_staged = W.self_staged, &done = W.done;
        std::vector<int32_t>&indeg = W.indeg, &queue = W.queue, &stamp = W.stamp;
        self_staged.resize(nm);
        for (int m = 0; m < nm; ++m) self_staged[m] = mv[m].staged;
        // If the staged pages of one pool do not fit the staging buffer, allow longer chains (fewer cuts).
        for (int max_level = x->kv_max_level;; max_level = std::min(kMaxLevelCap, max_level * 4)) {
          for (int m = 0; m < nm; ++m) mv[m].staged = self_staged[m];
          indeg.assign(nm, 0);
          done.assign(nm, 0);
          queue.clear();
          queue.reserve(nm);
          int n_direct = 0;
          for (int m = 0; m < nm; ++m) {
            mv[m].level = 0;
            if (mv[m].staged) { done[m] = 1; continue; }
            ++n_direct;
            for (int32_t e = blk_off[m]; e < blk_off[m + 1]; ++e) {
              if (mv[blk[e]].staged) mv[m].level = 1; else indeg[m]++;
            }
          }
          for (int m = 0; m < nm; ++m) if (!done[m] && indeg[m] == 0) queue.push_back(m);
          size_t qh = 0;
          int scan = 0, resolved = 0;
          stamp.assign(nm, -1);
          int32_t walk_id = 0;
          auto release = [&](int m, int lvl) {
            for (int32_t e = dep_off[m]; e < dep_off[m + 1]; ++e) {
              const int32_t d = dep[e];
              if (done[d] || mv[d].staged) continue;
              mv[d].level = std::max(mv[d].level, lvl);
              if (--indeg[d] == 0) queue.push_back(d);
            }
          };
          while (resolved < n_direct) {
            if (qh < queue.size()) {
              int m = queue[qh++];
              done[m] = 1;
              if (mv[m].level > max_level) {        // cut the chain here
                mv[m].staged = 1; --n_direct;
                release(m, 1);
              } else {
                ++resolved;
                release(m, mv[m].level + 1);
              }
              continue;
            }
            // only cycles (and what sits behind them) are left: walk blockers to find a node ON a cycle
            while (scan < nm && done[scan]) ++scan;
            int v = scan;
            ++walk_id;
            for (;;) {
              if (stamp[v] == walk_id) break;
              stamp[v] = walk_id;
              int nxt = -1;
              for (int32_t e = blk_off[v]; e < blk_off[v + 1]; ++e)
                if (!done[blk[e]] && !mv[blk[e]].staged) { nxt = blk[e]; break; }
              v = nxt;  // exists: indeg[v] > 0
            }
            mv[v].staged = 1; done[v] = 1; --n_direct;
            release(v, 1);
          }
          K = 0;
          int64_t ns = 0;
          for (int m = 0; m < nm; ++m) { if (!mv[m].staged) K = std::max(K, (int)mv[m].level); else ++ns; }
          if (ns * x->ep_page_bytes <= x->staging_bytes - x->w_stg_bytes || max_level >= kMaxLevelCap) break;
        }
      } else if (any_self) {
        // self-overlapping moves only: they are staged; nobody else depends on anything
        K = 0;
      }
      for (int m = 0; m < nm; ++m) if (mv[m].staged) mv[m].slot = n_staged++;
    }
    pools_per_group = n_pools_all;
    if (n_staged > 0) {
      int64_t per_pool = (int64_t)n_staged * x->ep_page_bytes;
      int64_t fit = (x->staging_bytes - x->w_stg_bytes) / per_pool;
      if (fit < 1) return MOEBIUS_E_STAGING;
      pools_per_group = (int)std::min<int64_t>(fit, n_pools_all);
      if (n_staged >= (1 << 24)) return MOEBIUS_E_STAGING;
    }
    n_pool_groups = nm > 0 ? (n_pools_all + pools_per_group - 1) / pools_per_group : 0;
    return MOEBIUS_OK;
  }

  // the plan object
  int new_plan() {
    // ---- build the plan ---------------------------------------------------------------------------
    P = new (std::nothrow) moebius_plan_t();
    if (!P) return MOEBIUS_E_INVAL;
    P->ctx = x; P->from = from; P->to = to; P->n_req = n_req;
    P->image = nullptr; P->tbl_image = nullptr; P->kv = nullptr; P->n_kv = 0; P->bt = nullptr;
    P->buf.p = nullptr; P->buf.bytes = 0; P->buf.pinned = false; P->buf.ev = nullptr;
    memset(&P->stats, 0, sizeof(P->stats));
    P->stats.struct_size = sizeof(moebius_stats_t);
    next_ctr = 0;
    return MOEBIUS_OK;
  }

  // ---- S2 (BASELINE.json north_star: "in-place permutation cycles through a bounded
  // staging buffer") -- one object whose EP view starts fewer slots behind its TP view than the object is
  // long, so that part of what it writes lands on its own unread source.
  // The object is cut into BLOCKS (rows [i*T, (i+1)*T) of EP rank q: contiguous on the EP side, R pieces
  // on the TP side).  Block b BLOCKS on block a when b's destination overlaps a's source and a has not
  // been read yet.  The blocks are executed in dependency WAVES: a wave holds every block all of whose
  // blockers were read in earlier waves.  When no block is ready (the permutation's cycles) the cheapest
  // blocked block is chosen and its blockers are PARKED: their source is saved into a staging slot
  // (EP->TP: the EP rows are copied there; TP->EP: the block is transposed INTO the slot) and finished
  // from the slot once their own destination is free; a slot is reused as soon as its block is finished.
  // `tmpl` carries the object's shape and unit geometry as weight_chain chose them.
  // The schedule of one in-place object: its blocks, the waves of the greedy simulation, and the shapes
  // its segments take.  stg_base / stg_bytes: the part of the weight staging area this object may use
  // (objects whose schedules run concurrently get disjoint parts).
  enum { OP_MOVE = 0, OP_FINISH = 1, OP_PARK = 2 };
  struct S2Op { int32_t blk, op, slot; };
  struct S2Sched {
    Seg tmpl, lsu;
    bool xt;
    int64_t T, rt, Rr, run, slot_bytes;
    int nb;
    int64_t first_slot;                    // where the object's slots start in the weight staging area (set by the caller)
    int peak_slots;                        // slots the schedule ever uses (they are handed out lowest first)
    std::vector<std::vector<S2Op>> waves;
  };

  struct S2Cached {
    int64_t run, rt, T, sS; int nb, n_slots, peak, n_parked; int64_t staged_bytes;
    std::vector<std::vector<S2Op>> waves;
  };
  std::vector<S2Cached> s2_cache;

  int s2_schedule(const Seg& tmpl_in, int64_t stg_bytes, S2Sched& sc) {
    Seg tmpl = tmpl_in;
    const int64_t run = tmpl.run_bytes, rt = tmpl.rows_total, Rr = (int64_t)R * run;
    const int64_t sS = (int64_t)x->ep_shift * x->S;            // EP view offset minus TP view offset
    const bool xt = seg_path(tmpl) == PATH_TMA && tmpl.groups_per_unit == tmpl.n_groups;
    // a tensor-map box cannot address the staging buffer: staged EP sides of short-run objects use ld/st
    Seg lsu = tmpl;
    if (xt) {
      lsu.kind = SEG_XPOSE;
      lsu.groups_per_unit = R; lsu.chunk_bytes = (uint32_t)run; lsu.chunks_per_run = 1;
      lsu.rows_per_unit = (uint32_t)std::max<int64_t>(1, unit_bytes / Rr);
    }
    // 2R+2 slots let the simulation below always make progress; with less staging it is tried with what
    // fits (it reports E_STAGING itself when a cycle needs more parked blocks than there are slots)
    int64_t unit_rows = xt ? tmpl.rows_per_unit : 1;
    int64_t t_max = stg_bytes / (2 * (int64_t)R + 2) / Rr;
    if (t_max < 1) t_max = std::min<int64_t>(1, stg_bytes / Rr);
    if (t_max < 1) return MOEBIUS_E_STAGING;
    if (xt && t_max < unit_rows) {       // blocks smaller than one box: the whole object goes through ld/st
      tmpl = lsu;
      unit_rows = 1;
    }
    int64_t T = (rt + kS2BlocksPerRank - 1) / kS2BlocksPerRank;
    T = (T + unit_rows - 1) / unit_rows * unit_rows;
    T = std::min(T, t_max / unit_rows * unit_rows);
    T = std::max<int64_t>(T, unit_rows);
    const int nb = (int)((rt + T - 1) / T), NB = nb * R;
    const int64_t slot_bytes = T * Rr;
    const int n_slots = (int)std::min<int64_t>(stg_bytes / slot_bytes, 1 << 20);
    auto rows_of = [&](int i) { return std::min<int64_t>(T, rt - (int64_t)i * T); };
    // objects of one shape have one schedule (every layer's gate and up, every layer's down): simulate once
    struct { int64_t run, rt, T, sS; int nb, n_slots; } key = {run, rt, T, sS, nb, n_slots};
    for (const S2Cached& c : s2_cache)
      if (c.run == key.run && c.rt == key.rt && c.T == key.T && c.sS == key.sS && c.nb == key.nb && c.n_slots == key.n_slots) {
        sc.waves = c.waves;
        P->stats.n_w_parked += c.n_parked;
        P->stats.w_staged_bytes += c.staged_bytes;
        sc.tmpl = tmpl; sc.lsu = lsu; sc.xt = xt;
        sc.T = T; sc.rt = rt; sc.Rr = Rr; sc.run = run; sc.slot_bytes = slot_bytes; sc.nb = nb; sc.first_slot = 0; sc.peak_slots = c.peak;
        return MOEBIUS_OK;
      }
    const int64_t staged_before = P->stats.w_staged_bytes;
    // blockers of every block (CSR): the blocks whose SOURCE this block's DESTINATION overlaps
    std::vector<int32_t> bo((size_t)NB + 1, 0), bl;
    std::vector<uint8_t> self((size_t)NB, 0);
    for (int q = 0; q < R; ++q) for (int i = 0; i < nb; ++i) {
      const int b = q * nb + i;
      int32_t tmp[160]; int nt = 0;
      auto note = [&](int a) { if (a == b) self[(size_t)b] = 1; else if (nt < 160) tmp[nt++] = a; };
      if (e2t) {     // writes TP rows [q*rt + i*T, +rows) on EVERY rank; sources: EP rows of rank j at sS + row*Rr
        const int64_t y0 = ((int64_t)q * rt + (int64_t)i * T) * run, y1 = y0 + rows_of(i) * run;
        if (y1 > sS && y0 < sS + rt * Rr) {
          const int64_t lo = std::max<int64_t>(0, (y0 - sS) / (T * Rr)), hi = std::min<int64_t>(nb - 1, (y1 - 1 - sS) / (T * Rr));
          for (int j = 0; j < R; ++j) for (int64_t a = (y0 < sS ? 0 : lo); a <= hi; ++a) note(j * nb + (int)a);
        }
      } else {       // writes EP rows [i*T, +rows) of rank q; sources: TP rows (global index q2*rt + row) read on every rank
        const int64_t w0 = sS + (int64_t)i * T * Rr, w1 = w0 + rows_of(i) * Rr;
        const int64_t g0 = w0 / run, g1 = std::min<int64_t>((w1 - 1) / run, (int64_t)R * rt - 1);
        for (int64_t g = g0; g <= g1;) {
          const int64_t q2 = g / rt, i2 = (g % rt) / T;
          note((int)(q2 * nb + i2));
          g = q2 * rt + std::min<int64_t>(rt, (i2 + 1) * T);     // first row of the next block
        }
      }
      std::sort(tmp, tmp + nt);
      nt = (int)(std::unique(tmp, tmp + nt) - tmp);
      for (int k = 0; k < nt; ++k) bl.push_back(tmp[k]);
      bo[(size_t)b + 1] = (int32_t)bl.size();
    }
    // Which blocks to park: a feedback vertex set F of the blocker graph (without F the graph has no cycle, so
    // parking only blocks of F always suffices).  Greedy: blocks that block themselves; then, as long as
    // pruning the blocks with no blocker or nothing blocked left among the rest does not empty it, the block
    // with the most (blockers x blocked).  For aliased views of a power-of-two shape the graph is the de
    // Bruijn graph on R-ary words of length 3 (block (q, a, b) is blocked by (j, q, a) for every j) and this
    // finds its minimum, the 176 necklaces of 512 words; taking the blockers of whichever block needs the
    // fewest parks, as round 2's first version did, parks 260-324.
    std::vector<uint8_t> inF((size_t)NB, 0);
    {
      std::vector<int32_t> so((size_t)NB + 1, 0), sl_;
      for (int b = 0; b < NB; ++b) for (int32_t e = bo[(size_t)b]; e < bo[(size_t)b + 1]; ++e) so[(size_t)bl[(size_t)e] + 1]++;
      for (int b = 0; b < NB; ++b) so[(size_t)b + 1] += so[(size_t)b];
      sl_.resize((size_t)so[(size_t)NB]);
      { std::vector<int32_t> pos(so.begin(), so.end() - 1);
        for (int b = 0; b < NB; ++b) for (int32_t e = bo[(size_t)b]; e < bo[(size_t)b + 1]; ++e) sl_[(size_t)pos[(size_t)bl[(size_t)e]]++] = b; }
      std::vector<uint8_t> alive((size_t)NB, 1);
      std::vector<int32_t> nin((size_t)NB, 0), nout((size_t)NB, 0);
      for (int b = 0; b < NB; ++b) if (self[(size_t)b]) { inF[(size_t)b] = 1; alive[(size_t)b] = 0; }
      for (int b = 0; b < NB; ++b) if (alive[(size_t)b]) {
        for (int32_t e = bo[(size_t)b]; e < bo[(size_t)b + 1]; ++e) nin[(size_t)b] += alive[(size_t)bl[(size_t)e]];
        for (int32_t e = so[(size_t)b]; e < so[(size_t)b + 1]; ++e) nout[(size_t)b] += alive[(size_t)sl_[(size_t)e]];
      }
      std::vector<int32_t> stack;
      auto kill = [&](int b) {           // b leaves the graph; neighbours that lose their last edge follow
        alive[(size_t)b] = 0;
        for (int32_t e = bo[(size_t)b]; e < bo[(size_t)b + 1]; ++e) { const int a = bl[(size_t)e]; if (alive[(size_t)a] && --nout[(size_t)a] == 0) stack.push_back(a); }
        for (int32_t e = so[(size_t)b]; e < so[(size_t)b + 1]; ++e) { const int a = sl_[(size_t)e]; if (alive[(size_t)a] && --nin[(size_t)a] == 0) stack.push_back(a); }
      };
      auto prune = [&]() {
        while (!stack.empty()) { const int b = stack.back(); stack.pop_back(); if (alive[(size_t)b]) kill(b); }
      };
      for (int b = 0; b < NB; ++b) if (alive[(size_t)b] && (nin[(size_t)b] == 0 || nout[(size_t)b] == 0)) stack.push_back(b);
      prune();
      for (;;) {
        int best = -1; int64_t best_w = -1;
        for (int b = 0; b < NB; ++b) if (alive[(size_t)b]) {
          const int64_t wgt = (int64_t)nin[(size_t)b] * nout[(size_t)b];
          if (wgt > best_w) { best_w = wgt; best = b; }
        }
        if (best < 0) break;
        inF[(size_t)best] = 1;
        kill(best);
        prune();
      }
    }
    // greedy wave simulation
    typedef S2Op Op;
    std::vector<std::vector<Op>>& waves = sc.waves;
    waves.clear();
    std::vector<int32_t> read_wave((size_t)NB, INT32_MAX);    // wave in which the block's source was read (moved or parked)
    std::vector<int32_t> slot_of((size_t)NB, -1);
    std::vector<uint8_t> done((size_t)NB, 0);
    std::vector<int32_t> free_slots;
    for (int k = n_slots - 1; k >= 0; --k) free_slots.push_back(k);
    int n_done = 0, n_parked = 0, peak = 0;
    // parks per stall: an eighth of the blocks -- against one block at a time that is 10 x fewer waves for the
    // same number of parked blocks (config 4's shapes: 128 -> 10-13 waves per object, 260-295 -> 271-324 parked)
    const int s2_batch = std::max(1, NB / 8);
    while (n_done < NB) {
      const int32_t w = (int32_t)waves.size();
      if (w > 4 * NB + 8) return MOEBIUS_E_STAGING;
      std::vector<Op> ops;
      std::vector<int32_t> freed;
      for (int b = 0; b < NB; ++b) {
        if (done[(size_t)b]) continue;
        if (self[(size_t)b] && !(slot_of[(size_t)b] >= 0 && read_wave[(size_t)b] < w)) continue;
        if (slot_of[(size_t)b] >= 0 && read_wave[(size_t)b] >= w) continue;     // parked in this very wave
        bool ok = true;
        for (int32_t e = bo[(size_t)b]; e < bo[(size_t)b + 1] && ok; ++e) ok = read_wave[(size_t)bl[(size_t)e]] < w;
        if (!ok) continue;
        if (slot_of[(size_t)b] >= 0) { ops.push_back({b, OP_FINISH, slot_of[(size_t)b]}); freed.push_back(slot_of[(size_t)b]); }
        else { ops.push_back({b, OP_MOVE, 0}); read_wave[(size_t)b] = w; }
        done[(size_t)b] = 1; ++n_done;
      }
      if (ops.empty()) {      // cycles: park the blockers of the blocks that need the fewest parks
        auto park = [&](int a) {
          const int32_t sl = free_slots.back(); free_slots.pop_back();
          peak = std::max(peak, sl + 1);
          slot_of[(size_t)a] = sl; read_wave[(size_t)a] = w;
          ops.push_back({a, OP_PARK, sl});
          ++n_parked;
          P->stats.w_staged_bytes += rows_of(a % nb) * Rr;
        };
        // One stall opens several blocks at once (s2_batch parks per wave at most): fewer, fatter waves.
        int parks = 0;
        do {
          // the block that needs the fewest parks among those whose unread blockers all belong to F (there is
          // always one while something is left: without F the graph is acyclic); any block as a last resort
          int best = -1, best_need = INT32_MAX, any = -1, any_need = INT32_MAX;
          for (int b = 0; b < NB; ++b) {
            if (done[(size_t)b]) continue;
            int need = (self[(size_t)b] && slot_of[(size_t)b] < 0) ? 1 : 0;
            bool in_f = true;
            for (int32_t e = bo[(size_t)b]; e < bo[(size_t)b + 1]; ++e) {
              const int a = bl[(size_t)e];
              if (read_wave[(size_t)a] == INT32_MAX) { ++need; in_f = in_f && inF[(size_t)a]; }
            }
            if (need <= 0) continue;
            if (in_f && need < best_need) { best = b; best_need = need; }
            if (need < any_need) { any = b; any_need = need; }
          }
          if (best < 0 && parks == 0) { best = any; best_need = any_need; }
          if (best < 0) break;
          if (best_need > (int)free_slots.size()) {
            if (parks == 0) return MOEBIUS_E_STAGING;
            break;
          }
          if (self[(size_t)best] && slot_of[(size_t)best] < 0) park(best);
          for (int32_t e = bo[(size_t)best]; e < bo[(size_t)best + 1]; ++e)
            if (read_wave[(size_t)bl[(size_t)e]] == INT32_MAX) park(bl[(size_t)e]);
          parks += best_need;
        } while (parks < s2_batch);
      }
      // freed slots go back so that the lowest index is handed out next (peak_slots stays the true peak)
      for (int32_t sl : freed) free_slots.push_back(sl);
      std::sort(free_slots.begin(), free_slots.end(), std::greater<int32_t>());
      waves.push_back(std::move(ops));
    }
    P->stats.n_w_parked += n_parked;
    s2_cache.push_back({run, rt, T, sS, nb, n_slots, peak, n_parked, P->stats.w_staged_bytes - staged_before, waves});
    sc.tmpl = tmpl; sc.lsu = lsu; sc.xt = xt;
    sc.T = T; sc.rt = rt; sc.Rr = Rr; sc.run = run; sc.slot_bytes = slot_bytes; sc.nb = nb; sc.first_slot = 0; sc.peak_slots = peak;
    return MOEBIUS_OK;
  }

  // Segments of ONE wave of a schedule: up to three kinds of work, full and ragged blocks apart (a segment
  // has one shape); every segment waits for (wait_ctr, wait_target) and signals ctr.  Returns the units added.
  uint32_t s2_emit_wave(const S2Sched& sc, size_t w, int wait_ctr, uint32_t wait_target, int ctr) {
    const Seg& tmpl = sc.tmpl; const Seg& lsu = sc.lsu;
    const bool xt = sc.xt;
    const int64_t T = sc.T, rt = sc.rt, Rr = sc.Rr, run = sc.run, slot_bytes = sc.slot_bytes;
    const int nb = sc.nb;
    auto rows_of = [&](int i) { return std::min<int64_t>(T, rt - (int64_t)i * T); };
    typedef S2Op Op;
    const std::vector<Op>& ops = sc.waves[w];
    uint32_t wave_units = 0;
    {
      for (int kind = 0; kind < 3; ++kind) for (int ragged = 0; ragged < 2; ++ragged) {
        const int64_t rows = ragged ? rows_of(nb - 1) : T;
        if (ragged && rows == T) continue;
        std::vector<WBlk> blks;
        for (const Op& o : ops) {
          const int i = o.blk % nb;
          if (o.op != kind || (rows_of(i) != T) != (ragged != 0)) continue;
          blks.push_back({(uint32_t)(o.blk / nb), (uint32_t)((int64_t)i * T), (uint32_t)rows_of(i), (uint32_t)(sc.first_slot + o.slot)});
        }
        if (blks.empty()) continue;
        // which side of the work is plain copying between the EP rows and the slot
        const bool copy = (kind == OP_PARK && e2t) || (kind == OP_FINISH && !e2t);
        Seg t;
        if (!copy) {
          // a parked block's EP side is its staging slot: on the TMA path the TP-side box serves it (the EP side
          // is then one bulk copy from / into the slot), which needs whole boxes; ragged rows go through ld/st
          const bool box_ok = xt && seg_path(tmpl) == PATH_TMA && rows % (int64_t)tmpl.rows_per_unit == 0;
          t = (kind == OP_MOVE || !xt || box_ok) ? tmpl : lsu;
          t.kv_mode = kind == OP_MOVE ? 0u : 1u;             // 1: the EP side of every block is its staging slot
          t.stg_pools = 0;                                    // an irregular list: WBlk descriptors
          t.pool_begin = (uint32_t)P->wblk.size();
          t.n_desc = (uint32_t)blks.size();
          t.pool_bytes = slot_bytes;
          const uint32_t rbpb = (uint32_t)((rows + t.rows_per_unit - 1) / t.rows_per_unit);
          t.pools_per_unit = rbpb * (t.n_groups / t.groups_per_unit) * t.chunks_per_run;
          t.n_units = t.n_desc * t.pools_per_unit;
          for (const WBlk& k : blks) P->wblk.push_back(k);
        } else {
          t = blank_seg();
          t.kind = SEG_BULK | ((x->use_tma ? PATH_TMA : PATH_LSU) << 8);
          t.kv_mode = e2t ? 2u : 1u;                           // EP->TP park: destination in staging; TP->EP finish: source
          t.ep_is_src = e2t;
          t.rows_total = (uint32_t)(rows * R);                 // the block's EP rows as R*rows contiguous runs
          t.run_bytes = (uint32_t)run;
          const int64_t lim = x->use_tma ? x->stage_bytes : unit_bytes;
          t.chunk_bytes = pick_chunk(run, lim);
          t.chunks_per_run = (uint32_t)(run / t.chunk_bytes);
          t.rows_per_unit = t.chunks_per_run == 1 ? (uint32_t)std::max<int64_t>(1, std::min<int64_t>(rows * R, lim / run)) : 1;
          t.row_blocks = (t.rows_total + t.rows_per_unit - 1) / t.rows_per_unit;
          t.ep_off = run; t.tp_off = run;
          t.desc_begin = (uint32_t)P->bulk.size();
          t.n_desc = (uint32_t)blks.size();
          for (const WBlk& k : blks) {
            const int64_t ep = (int64_t)k.q * x->rank_stride + tmpl.ep_off + (int64_t)k.row0 * Rr;
            const int64_t sl = (int64_t)k.slot * slot_bytes;
            P->bulk.push_back(e2t ? BulkDesc{ep, sl} : BulkDesc{sl, ep});
          }
          t.n_units = t.n_desc * t.row_blocks * t.chunks_per_run;
        }
        t.wait_ctr = wait_ctr; t.wait_target = wait_target;
        t.signal_ctr = ctr;
        wave_units += t.n_units;
        push_seg(cw, t);
      }
    }
    return wave_units;
  }

  // One in-place object on its own: its waves one after the other, behind (prev_ctr, prev_units).
  int s2_object(const Seg& tmpl_in, int& prev_ctr, uint32_t& prev_units) {
    S2Sched sc;
    if (int rc = s2_schedule(tmpl_in, x->w_stg_bytes, sc)) return rc;
    P->stats.n_w_waves += (int32_t)sc.waves.size();
    for (size_t w = 0; w < sc.waves.size(); ++w) {
      if (next_ctr >= (uint32_t)kMaxCounters) return MOEBIUS_E_STAGING;
      const int ctr = (int)next_ctr++;
      const uint32_t units = s2_emit_wave(sc, w, prev_ctr, prev_units, ctr);
      prev_ctr = ctr; prev_units = units;
    }
    return MOEBIUS_OK;
  }

  // Aliased views (shift 0): an object's move stays inside its own slot, so the objects do not depend on one
  // another and their schedules run side by side -- wave w of every object of a group is ONE dependency
  // level of the launch -- each object parking into its own part of the staging area.  A group is as many
  // consecutive objects as the staging area holds at the peak of their schedules.
  int s2_objects_concurrent(const std::vector<Seg>& tmpls) {
    // every object is scheduled as if it were alone (same blocks, same waves as on its own); what it needs
    // of the staging area is the peak of slots its schedule ever holds
    std::vector<S2Sched> sc(tmpls.size());
    for (size_t o = 0; o < tmpls.size(); ++o)
      if (int rc = s2_schedule(tmpls[o], x->w_stg_bytes, sc[o])) return rc;
    int prev_ctr = -1; uint32_t prev_units = 0;
    for (size_t o0 = 0; o0 < sc.size();) {
      size_t n = 0;
      int64_t end = 0;
      while (o0 + n < sc.size()) {
        S2Sched& c = sc[o0 + n];
        const int64_t first = (end + c.slot_bytes - 1) / c.slot_bytes;
        const int64_t e = (first + std::max(1, c.peak_slots)) * c.slot_bytes;
        if (n > 0 && e > x->w_stg_bytes) break;
        c.first_slot = first;
        end = e;
        ++n;
      }
      // Inside a group every object runs its own chain of waves (its own counters): the segments are laid
      // out wave by wave across the objects, so by the time a pipe reaches wave w+1 of an object the other
      // objects' wave-w units have been handed out in between and its wave w is long complete -- no
      // device-wide drain per wave.  Only the groups are separated: the last wave of every object signals
      // the group's counter, and the next group, which reuses the staging area, waits for all of it.
      size_t n_waves = 0;
      for (size_t k = 0; k < n; ++k) n_waves = std::max(n_waves, sc[o0 + k].waves.size());
      P->stats.n_w_waves += (int32_t)n_waves;
      if (next_ctr >= (uint32_t)kMaxCounters) return MOEBIUS_E_STAGING;
      const int group_ctr = (int)next_ctr++;
      uint32_t group_units = 0;
      std::vector<int> o_ctr(n, prev_ctr);
      std::vector<uint32_t> o_units(n, prev_units);
      for (size_t w = 0; w < n_waves; ++w)
        for (size_t k = 0; k < n; ++k) {
          const S2Sched& c = sc[o0 + k];
          if (w >= c.waves.size()) continue;
          const bool last = w + 1 == c.waves.size();
          int ctr = group_ctr;
          if (!last) {
            if (next_ctr >= (uint32_t)kMaxCounters) return MOEBIUS_E_STAGING;
            ctr = (int)next_ctr++;
          }
          const uint32_t units = s2_emit_wave(c, w, o_ctr[k], o_units[k], ctr);
          if (last) group_units += units;
          o_ctr[k] = ctr; o_units[k] = units;
        }
      prev_ctr = group_ctr; prev_units = group_units;
      o0 += n;
    }
    return MOEBIUS_OK;
  }

  // expert-weight objects
  int weight_chain() {
    // weights: one segment per (layer, matrix) object, chained in the direction-specific order
    // ("EP->TP adopts the sequential order while TP->EP adopts the reverse order").
    // Every EP view starts ep_shift slots (= the largest object) behind its TP view, so an object's
    // write never lands on its own source nor on the source of an object still to come, and the
    // regions it does overwrite belong to objects earlier in the chain, which have completed
    // (each link waits for the previous one, transitively for all of them).
    if (R > 1) {
      const int n_links = L * x->n_obj;
      // shape, data path and unit geometry of one chain link
      auto link_seg = [&](const WObj& ob, int tp_slot, Seg& s) -> int {
        s = blank_seg();
        s.kind = SEG_XPOSE;
        s.ep_is_src = e2t;
        s.n_groups = R;
        s.rep = 1;
        int64_t run = !ob.long_run ? (int64_t)(c.I / R) * x->wb : (int64_t)(c.I / R) * c.H * x->wb;
        s.rows_total = !ob.long_run ? (uint32_t)(c.E / R) * c.H : (uint32_t)(c.E / R) * ob.row_mult;
        if (run > (1ll << 31)) return MOEBIUS_E_INVAL;
        s.run_bytes = (uint32_t)run;
        s.desc_begin = (uint32_t)(tp_slot + x->ep_shift);   // EP slot index (tensor-map coordinate)
        const int64_t stage = x->stage_bytes;
        const uint32_t lt_chunk = pick_chunk(run, stage);
        if (x->use_tma && !ob.long_run && x->xt_ok) {
          // one tensor-map box per unit: xt_rows rows x all R groups
          s.kind = SEG_XPOSE | (PATH_TMA << 8);
          s.groups_per_unit = R;
          s.chunk_bytes = (uint32_t)run;
          s.chunks_per_run = 1;
          s.rows_per_unit = (uint32_t)x->xt_rows;
        } else if (x->use_tma && (run > 1024 || run * R > stage) && (lt_chunk == run || lt_chunk >= 4096)) {
          // one group per unit: plain bulk copies (long runs: the down projection, the W13 stack)
          s.kind = SEG_XPOSE | (PATH_TMA << 8);
          s.groups_per_unit = 1;
          s.chunk_bytes = lt_chunk;
          s.chunks_per_run = (uint32_t)(run / s.chunk_bytes);
          s.rows_per_unit = s.chunks_per_run == 1 ? (uint32_t)std::min<int64_t>(32, std::max<int64_t>(1, stage / run)) : 1;
        } else if (run * R <= unit_bytes || run <= 4096) {
          s.groups_per_unit = R;
          s.chunk_bytes = (uint32_t)run;
          s.chunks_per_run = 1;
          s.rows_per_unit = (uint32_t)std::max<int64_t>(1, unit_bytes / (run * R));
        } else {
          s.groups_per_unit = 1;
          s.chunk_bytes = pick_chunk(run, unit_bytes);
          s.chunks_per_run = (uint32_t)(run / s.chunk_bytes);
          s.rows_per_unit = s.chunks_per_run == 1 ? (uint32_t)std::max<int64_t>(1, unit_bytes / run) : 1;
        }
        s.row_blocks = (s.rows_total + s.rows_per_unit - 1) / s.rows_per_unit;
        s.tp_off = x->w_off + (int64_t)tp_slot * x->S;
        s.ep_off = x->w_off + (int64_t)(tp_slot + x->ep_shift) * x->S;
        int64_t nu = (int64_t)R * s.row_blocks * (s.n_groups / s.groups_per_unit) * s.chunks_per_run;
        if (nu > (1ll << 30)) return MOEBIUS_E_INVAL;
        s.n_units = (uint32_t)nu;
        return MOEBIUS_OK;
      };
      // Banded chain (equal-sized objects, every move out of place): a link conflicts only with its
      // predecessor, whose source slot it overwrites, and only half by half -- the bytes a unit writes
      // in the first half of the slot were read by the predecessor's units of the first half of the
      // rows (EP->TP; TP->EP mirrored).  Each link is therefore cut into 2 x 2 segments (half of the EP
      // ranks x half of the rows, as block lists) with one counter per half: a segment waits for ONE
      // half of the predecessor and the links overlap by a quarter, so no device-wide drain separates
      // them.  OFF by default (moebius_set_chain_bands): measured on B200 it removes every stall (0 pipes
      // ever wait, against 296 per link) and is still 9-13 % SLOWER at the 30B shape (weight-only switch
      // 2.57 ms vs 2.30 ms at L = 6) -- the quarter-object order itself costs more than the drains it
      // saves, even with the waits switched off (2.50 ms); DESIGN.md section 3.
      bool band = x->chain_bands && x->n_obj == 3 && x->ep_shift == 1 && R % 2 == 0;
      for (int o = 0; o < x->n_obj && band; ++o) {
        Seg t;
        if (int rc = link_seg(x->obj[o], x->obj[o].slot, t)) return fail(rc);
        band = t.rows_total % 2 == 0 && (t.rows_total / 2) % t.rows_per_unit == 0;
      }
      int prev_ctr = -1; uint32_t prev_units = 0;
      int band_ctr[2] = {-1, -1}; uint32_t band_units[2] = {0, 0};
      if (x->ep_shift == 0) {       // aliased views: independent objects, their in-place schedules side by side
        std::vector<Seg> tmpls((size_t)n_links);
        for (int step = 0; step < n_links; ++step) {
          const int k = e2t ? step : n_links - 1 - step;
          const WObj& ob = x->obj[k % x->n_obj];
          if (int rc = link_seg(ob, 3 * (k / x->n_obj) + ob.slot, tmpls[(size_t)step])) return fail(rc);
        }
        if (int rc = s2_objects_concurrent(tmpls)) return fail(rc);
      }
      for (int step = 0; step < n_links && x->ep_shift > 0; ++step) {
        const int k = e2t ? step : n_links - 1 - step;
        const int layer = k / x->n_obj;
        const WObj& ob = x->obj[k % x->n_obj];
        const int tp_slot = 3 * layer + ob.slot;
        Seg s;
        if (int rc = link_seg(ob, tp_slot, s)) return fail(rc);
        if (band) {
          if (next_ctr + 2 > (uint32_t)kMaxCounters) return fail(MOEBIUS_E_INVAL);
          const int ctr[2] = {(int)next_ctr, (int)next_ctr + 1};
          next_ctr += 2;
          uint32_t sig_units[2] = {0, 0};
          const uint32_t half = s.rows_total / 2;
          for (int i = 0; i < 4; ++i) {
            const int wi = i / 2, oi = i % 2;          // ordered by the half they wait for
            const int qh = e2t ? wi : oi, rh = e2t ? oi : wi;   // half of the EP ranks, half of the rows
            const int sig = e2t ? rh : qh;              // as a SOURCE: EP->TP read by rows, TP->EP by TP offset (= rank half)
            Seg t = s;
            t.n_desc = (uint32_t)(R / 2);                 // a regular block list: rows [rh*half, +half) of ranks qh*R/2 ...
            t.stg_pools = 1; t.stg_pool_begin = (uint32_t)(qh * (R / 2));
            t.pool_begin = (uint32_t)rh * half; t.n_pools = half;
            t.pools_per_unit = ((half + t.rows_per_unit - 1) / t.rows_per_unit) * (t.n_groups / t.groups_per_unit) * t.chunks_per_run;
            t.n_units = t.n_desc * t.pools_per_unit;
            t.kv_mode = 0; t.pool_bytes = 0;
            t.wait_ctr = band_ctr[wi]; t.wait_target = band_units[wi];
            t.signal_ctr = ctr[sig];
            sig_units[sig] += t.n_units;
            push_seg(cw, t);
          }
          band_ctr[0] = ctr[0]; band_ctr[1] = ctr[1];
          band_units[0] = sig_units[0]; band_units[1] = sig_units[1];
          continue;
        }
        if (ob.n_slots > x->ep_shift) {      // its EP view overlaps its own TP view: the in-place path (S2)
          if (int rc = s2_object(s, prev_ctr, prev_units)) return fail(rc);
          continue;
        }
        s.wait_ctr = prev_ctr; s.wait_target = prev_units;
        if (next_ctr >= (uint32_t)kMaxCounters) return fail(MOEBIUS_E_INVAL);   // the counters sit below the uploaded image
        s.signal_ctr = (int32_t)next_ctr++;
        prev_ctr = s.signal_ctr; prev_units = s.n_units;
        push_seg(cw, s);
      }
      int64_t all = (int64_t)3 * L * c.E * c.H * c.I * x->wb;
      P->stats.w_relocated = P->stats.w_read = all;
      P->stats.w_moved = all / R * (R - 1);
    }
    return MOEBIUS_OK;
  }

  // fp8 block scales
  int scale_copies() {
    // fp8 block scales: TP and EP scale views live in disjoint fixed regions, so these are plain
    // out-of-place 2-D copies with no hazard (reading A13)
    if (c.w_dtype == MOEBIUS_FP8_E4M3_B128) {   // also for R == 1: the two scale views never alias
      const int HB = c.H / 128, IB = c.I / 128, EL = c.E / R;
      for (int l = 0; l < L; ++l) for (int m = 0; m < x->n_obj; ++m) {
        const WObj& ob = x->obj[m];
        int64_t tp_within = 0, ep_within = 0;
        for (int mm = 0; mm < m; ++mm) { tp_within += x->sg[mm].tp_bytes; ep_within += x->sg[mm].ep_bytes; }
        int prev_hi = 0;
        for (int j = 0; j < R; ++j) {
          int lo, hi; scale_blocks(j, R, c.I, &lo, &hi);
          int nb = hi - lo;
          int a = e2t ? lo : std::max(lo, prev_hi);   // TP->EP: each EP block is read from its lowest holder
          const int fresh_hi = prev_hi;               // blocks below it were already counted as read
          prev_hi = std::max(prev_hi, hi);
          int take = hi - a;
          if (take <= 0) continue;
          for (int q = 0; q < R; ++q) {
            C2dDesc d;
            int64_t tp_base = (int64_t)j * x->rank_stride + x->scale_tp_off + l * x->scale_tp_layer + tp_within;
            int64_t ep_base = (int64_t)q * x->rank_stride + x->scale_ep_off + l * x->scale_ep_layer + ep_within;
            int64_t tp_o, ep_o; uint32_t rows, run, tp_st, ep_st;
            if (!ob.long_run) {   // TP [E, HB, nb] ; EP [EL, HB, IB]; rows = (e', hb)
              rows = (uint32_t)EL * HB; run = (uint32_t)take * 4;
              tp_st = (uint32_t)nb * 4; ep_st = (uint32_t)IB * 4;
              tp_o = tp_base + ((int64_t)q * EL * HB * nb + (a - lo)) * 4;
              ep_o = ep_base + (int64_t)a * 4;
            } else {       // TP [E, mult*nb, HB] ; EP [EL, mult*IB, HB]; rows = (e', gate|up block)
              const int mult = ob.row_mult;
              rows = (uint32_t)EL * mult; run = (uint32_t)take * HB * 4;
              tp_st = (uint32_t)nb * HB * 4; ep_st = (uint32_t)IB * HB * 4;
              tp_o = tp_base + ((int64_t)q * EL * mult * nb + (a - lo)) * HB * 4;
              ep_o = ep_base + (int64_t)a * HB * 4;
            }
            d.rows = rows; d.run_bytes = run;
            if (e2t) { d.src_off = ep_o; d.dst_off = tp_o; d.src_stride = ep_st; d.dst_stride = tp_st; }
            else     { d.src_off = tp_o; d.dst_off = ep_o; d.src_stride = tp_st; d.dst_stride = ep_st; }
            P->c2d.push_back(d);
            int64_t bytes = (int64_t)rows * run;
            P->stats.w_relocated += bytes;
            if (q != j) P->stats.w_moved += bytes;
            // unique source bytes (reading A15): EP->TP reads a straddled block once for both holders
            const int fresh = hi - std::max(lo, fresh_hi);
            if (fresh > 0) P->stats.w_read += (int64_t)rows * fresh * (run / take);
          }
        }
      }
      Seg s = blank_seg();
      s.kind = SEG_COPY2D;
      s.ep_is_src = e2t;          // which side of a descriptor is the EP side (rank-share filter)
      s.desc_begin = 0;
      s.n_desc = (uint32_t)P->c2d.size();
      s.n_units = s.n_desc;
      push_seg(cs, s);
    }
    return MOEBIUS_OK;
  }

  // attention projections
  int attention_copies() {
    // MOEBIUS_ATTN_DUAL: both layouts are resident, the switch is a pointer swap -- nothing to do.
    // MOEBIUS_ATTN_GATHER: a rank's head shard sits in place inside its full-size tensor, so EP->TP
    // keeps the local slice (nothing moves) and TP->EP rebuilds the full projections from the other
    // ranks' shards: the paper's All-Gather, here one pulled copy per (layer, tensor, receiver, head
    // block).  Sources (a rank's own shard) are never written by this switch: no hazard, no ordering.
    if (c.attn_mode != MOEBIUS_ATTN_GATHER || e2t || R == 1) return MOEBIUS_OK;
    const int Hq = c.n_q_heads, D = c.head_dim, Hkv = c.kv_heads;
    const int64_t head = (int64_t)D * c.H * 2, stage = x->stage_bytes;
    for (int a = 0; a < 4; ++a) {
      const bool kv = a == 1 || a == 2;
      Seg s = blank_seg();
      s.kind = SEG_BULK | ((x->use_tma ? PATH_TMA : PATH_LSU) << 8);
      s.ep_is_src = 0;
      s.desc_begin = (uint32_t)P->bulk.size();
      int64_t run, rows, stride;
      if (a == 3) { rows = c.H; run = (int64_t)(Hq / R) * D * 2; stride = (int64_t)Hq * D * 2; }   // wo: column block per row
      else        { rows = 1; run = (kv ? (int64_t)x->hpr : (int64_t)(Hq / R)) * head; stride = run; }
      s.rows_total = (uint32_t)rows;
      s.run_bytes = (uint32_t)std::min<int64_t>(run, UINT32_MAX);
      s.chunk_bytes = pick_chunk(run, x->use_tma ? stage : unit_bytes);
      s.chunks_per_run = (uint32_t)(run / s.chunk_bytes);
      s.rows_per_unit = s.chunks_per_run == 1 ? (uint32_t)std::max<int64_t>(1, std::min<int64_t>(rows, (x->use_tma ? stage : unit_bytes) / run)) : 1;
      s.row_blocks = (uint32_t)((rows + s.rows_per_unit - 1) / s.rows_per_unit);
      s.ep_off = stride; s.tp_off = stride;     // BULK: source / destination row strides
      for (int l = 0; l < L; ++l) {
        const int64_t lbase = x->attn_off + (int64_t)l * x->attn_layer_bytes + x->attn_full_off[a];
        for (int q = 0; q < R; ++q) {
          // blocks of the head axis, one per TP holder: block b is read from its lowest-rank holder
          const int n_blocks = kv ? (Hkv >= R ? R : Hkv) : R;
          for (int b = 0; b < n_blocks; ++b) {
            const int src = kv && Hkv < R ? b * x->rep : b;            // lowest holder (the rule of reading A5)
            const bool held = kv && Hkv < R ? (q / x->rep == b) : (q == b);
            if (held) continue;                                         // already in place on rank q
            const int64_t within = a == 3 ? (int64_t)b * run : (int64_t)b * run;
            BulkDesc d;
            d.src_off = (int64_t)src * x->rank_stride + lbase + within;
            d.dst_off = (int64_t)q * x->rank_stride + lbase + within;
            P->bulk.push_back(d);
            P->stats.attn_moved += rows * run; P->stats.attn_relocated += rows * run; P->stats.attn_read += rows * run;
          }
        }
      }
      s.n_desc = (uint32_t)P->bulk.size() - s.desc_begin;
      const int64_t nu = (int64_t)s.n_desc * s.row_blocks * s.chunks_per_run;
      if (nu > (1ll << 30)) return fail(MOEBIUS_E_INVAL);
      s.n_units = (uint32_t)nu;
      push_seg(ca, s);
    }
    return MOEBIUS_OK;
  }

  // KV rounds as segments + byte accounting
  int kv_segments() {
    // KV: descriptors ordered [level 0][level 1]...[level K][staged]
    if (nm > 0) {
      std::vector<uint32_t>& lvl_begin = W.lvl_begin;
      lvl_begin.assign(K + 2, 0);
      for (int m = 0; m < nm; ++m) if (!mv[m].staged) lvl_begin[mv[m].level + 1]++;
      for (int l = 0; l <= K; ++l) lvl_begin[l + 1] += lvl_begin[l];
      const uint32_t n_direct = lvl_begin[K + 1];   // the descriptors themselves are written into the image below
      const uint32_t ppu_lsu = (uint32_t)std::max<int64_t>(1, std::min<int64_t>(unit_bytes / x->ep_page_bytes, 2));
      const bool kv_tma = x->use_tma && x->kt_ok;
      uint32_t ppu = kv_tma ? (uint32_t)x->kt_pools : ppu_lsu;
      auto kv_seg = [&](uint32_t mode, uint32_t ep_src, uint32_t d0, uint32_t nd, int pool0, int npool) {
        Seg s = blank_seg();
        const bool tma = kv_tma;   // staged pages too: the staging buffer has its own tensor map (page images)
        (void)mode;
        const uint32_t ppu = tma ? (uint32_t)x->kt_pools : ppu_lsu;
        s.kind = SEG_KV | ((tma ? PATH_TMA : PATH_LSU) << 8);
        s.kv_mode = mode;
        s.ep_is_src = ep_src;
        s.run_bytes = (uint32_t)x->run_kv;
        s.n_groups = (uint32_t)x->G;
        s.rep = (uint32_t)x->rep;
        s.ep_off = s.tp_off = x->kv_off;
        s.desc_begin = d0; s.n_desc = nd;
        s.pool_begin = (uint32_t)pool0; s.n_pools = (uint32_t)npool;
        s.pools_per_unit = std::min<uint32_t>(ppu, (uint32_t)npool);
        s.ep_page_bytes = (uint32_t)x->ep_page_bytes;
        s.tp_page_bytes = (uint32_t)x->tp_page_bytes;
        s.pool_bytes = x->pool_bytes;
        s.stg_pool_begin = (uint32_t)pool0;
        s.stg_pools = (uint32_t)npool;
        uint32_t pool_blocks = (s.n_pools + s.pools_per_unit - 1) / s.pools_per_unit;
        s.n_units = nd * pool_blocks;
        return s;
      };
      // a round = every segment that signals the same counter; the next round waits for all of them
      const int64_t kv_units_est = (int64_t)nm * ((n_pools_all + ppu - 1) / ppu);
      // KV work is cut into slices that the merge interleaves with the weight chain, so that a link's
      // drain hides behind independent KV units: one slice per link, but no slice under 2,048 units
      // (moebius_set_kv_slice sets the floor).  Since a segment change costs a pipe one round trip instead of
      // a binary search, 2,048 beats the earlier 8,192: config 2 - 7 %, 30B - 0.6 %, 235B and fp8 unchanged.
      const int64_t slice_floor = x->kv_slice_floor > 0 ? x->kv_slice_floor : 2048;
      const int64_t slice_units = std::max<int64_t>(slice_floor, kv_units_est / std::max(1, 3 * L));
      int prev_ctr = -1; uint32_t prev_total = 0;
      for (int g = 0; g < n_pool_groups; ++g) {
        int pool0 = g * pools_per_group;
        int npool = std::min(pools_per_group, n_pools_all - pool0);
        for (int round = 0; round <= K + 1; ++round) {
          std::vector<Seg> parts;
          if (round == 0 && n_staged)      // save staged sources: EP->TP copies the EP page, TP->EP gathers into the slot
            parts.push_back(kv_seg(e2t ? KV_STG_COPY : KV_MOVE_STG, e2t ? 1u : 0u, n_direct, (uint32_t)n_staged, pool0, npool));
          if (round <= K && lvl_begin[round + 1] > lvl_begin[round])
            parts.push_back(kv_seg(KV_MOVE, e2t ? 1u : 0u, lvl_begin[round], lvl_begin[round + 1] - lvl_begin[round], pool0, npool));
          if (round == K + 1 && n_staged)  // every source has been read by now
            parts.push_back(kv_seg(e2t ? KV_MOVE_STG : KV_STG_COPY, e2t ? 1u : 0u, n_direct, (uint32_t)n_staged, pool0, npool));
          uint32_t total = 0;
          for (auto& s : parts) total += s.n_units;
          if (!total) continue;
          if (next_ctr >= (uint32_t)kMaxCounters) return fail(MOEBIUS_E_STAGING);
          int ctr = (int)next_ctr++;
          for (auto& s : parts) {
            // slice long segments so they interleave with the weight chain (drains of one hide behind the other)
            uint32_t pool_blocks = (s.n_pools + s.pools_per_unit - 1) / s.pools_per_unit;
            uint32_t desc_per_slice = (uint32_t)std::max<int64_t>(1, slice_units / pool_blocks);
            for (uint32_t d0 = 0; d0 < s.n_desc; d0 += desc_per_slice) {
              Seg t = s;
              t.desc_begin = s.desc_begin + d0;
              t.n_desc = std::min(desc_per_slice, s.n_desc - d0);
              t.n_units = t.n_desc * pool_blocks;
              t.wait_ctr = prev_ctr; t.wait_target = prev_total;
              t.signal_ctr = ctr;
              push_seg(ck, t);
            }
          }
          prev_ctr = ctr; prev_total = total;
        }
      }
      // accounting (reading A15): per pool, per move
      for (int m = 0; m < nm; ++m) {
        int64_t row = (int64_t)mv[m].ntok * x->run_kv;     // one group's bytes of this page
        if (e2t) {
          P->stats.kv_read += row * x->G;
          P->stats.kv_relocated += row * x->G * x->rep;
          P->stats.kv_moved += row * (x->G * x->rep - 1);  // the owner's own shard stays on its rank
        } else {
          P->stats.kv_read += row * x->G;
          P->stats.kv_relocated += row * x->G;
          P->stats.kv_moved += row * (x->G - 1);           // the new owner always holds one group itself
        }
      }
      P->stats.kv_read *= n_pools_all; P->stats.kv_relocated *= n_pools_all; P->stats.kv_moved *= n_pools_all;
    }
    return MOEBIUS_OK;
  }

  // one ordered list; dependency waves
  int merge_and_waves() {
    // merge the chains by fractional position (each keeps its own order)
    struct Item { double pos; int chain; size_t idx; };
    std::vector<Item> items;
    auto add_chain = [&](Chain& ch, int id) {
      int64_t acc = 0;
      for (size_t i = 0; i < ch.segs.size(); ++i) {
        items.push_back({ch.units ? (acc + 0.5 * ch.segs[i].n_units) / (double)ch.units : 0.0, id, i});
        acc += ch.segs[i].n_units;
      }
    };
    add_chain(cs, 0); add_chain(cw, 1); add_chain(ck, 2); add_chain(ca, 3);
    std::stable_sort(items.begin(), items.end(), [](const Item& a, const Item& b) {
      if (a.chain == 0 || b.chain == 0) return a.chain == 0 && b.chain != 0;
      return a.pos < b.pos;
    });
    ub = 0;
    for (auto& it : items) {
      Seg s = (it.chain == 0 ? cs : it.chain == 1 ? cw : it.chain == 2 ? ck : ca).segs[it.idx];
      s.unit_begin = (uint32_t)ub;
      ub += s.n_units;
      P->segs.push_back(s);
    }
    if (ub >= (1ull << 32) || P->segs.size() > (size_t)kMaxSegs || (int64_t)nm > x->max_kv_desc ||
        P->c2d.size() > (size_t)x->max_c2d || P->bulk.size() > (size_t)(x->max_bulk + x->max_wblk) ||
        P->wblk.size() > (size_t)x->max_wblk)
      return fail(MOEBIUS_E_INVAL);
    P->total_units = (uint32_t)ub;
    P->n_counters = next_ctr;
    P->uses_tma = false;
    for (const Seg& s : P->segs) if (seg_path(s) == PATH_TMA) P->uses_tma = true;
    P->stage_bytes = x->stage_bytes;
    P->xt_rows = x->xt_rows;

    // Waves: wave(s) = 0 without a dependency, else 1 + the latest wave among the segments that signal
    // the counter s waits on.  A multi-GPU run executes wave by wave with a barrier across GPUs in
    // between (one barrier per dependency round); the fused launch ignores them.
    std::vector<int32_t>& seg_wave = P->seg_wave;
    seg_wave.assign(P->segs.size(), 0);
    {
      std::vector<int32_t> ctr_wave(next_ctr ? next_ctr : 1, -1);
      int32_t n_waves = P->segs.empty() ? 0 : 1;
      for (size_t i = 0; i < P->segs.size(); ++i) {
        const Seg& sg = P->segs[i];
        int32_t w = sg.wait_ctr >= 0 ? ctr_wave[(size_t)sg.wait_ctr] + 1 : 0;
        seg_wave[i] = w;
        if (sg.signal_ctr >= 0) ctr_wave[(size_t)sg.signal_ctr] = std::max(ctr_wave[(size_t)sg.signal_ctr], w);
        n_waves = std::max(n_waves, w + 1);
      }
      P->n_waves = n_waves;
    }
    return MOEBIUS_OK;
  }

  // upload images
  int build_images() {
    const std::vector<int32_t>& seg_wave = P->seg_wave;
    // ---- target request state + upload images (written in place: [segs][kv][c2d][waves] | tables) ---
    P->lens.assign(seq_lens, seq_lens + n_req);
    P->owner = owner;
    int64_t seg_b = align_up((int64_t)P->segs.size() * sizeof(Seg), 256);
    int64_t kv_b = align_up((int64_t)nm * sizeof(KvDesc), 256);
    int64_t c2d_b = align_up((int64_t)P->c2d.size() * sizeof(C2dDesc), 256);
    const int64_t hdr_b = sizeof(PlanHdr);
    int64_t bulk_b = align_up((int64_t)P->bulk.size() * sizeof(BulkDesc), 256);
    int64_t wblk_b = align_up((int64_t)P->wblk.size() * sizeof(WBlk), 256);
    P->kv_img_off = hdr_b + seg_b;
    P->c2d_img_off = hdr_b + seg_b + kv_b;
    P->bulk_img_off = hdr_b + seg_b + kv_b + c2d_b;
    P->wblk_img_off = hdr_b + seg_b + kv_b + c2d_b + bulk_b;
    P->wave_img_off = hdr_b + seg_b + kv_b + c2d_b + bulk_b + wblk_b;
    const int64_t wave_b = (int64_t)P->n_waves * hdr_b + (int64_t)P->segs.size() * (int64_t)sizeof(Seg);
    P->wave_tab_img_off = P->wave_img_off + wave_b;
    P->image_bytes = P->wave_tab_img_off + align_up((int64_t)P->n_waves * 4, 256);
    if (kSegOff + P->image_bytes > x->desc_bytes) return fail(MOEBIUS_E_INVAL);
    P->tbl_bytes = 4 * ((int64_t)kTblHdrInts + 2 * (int64_t)c.max_requests + (int64_t)n_req * MP);
    if (!image_acquire(x, P->image_bytes + P->tbl_bytes + 256, &P->buf)) return fail(MOEBIUS_E_INVAL);
    P->image = P->buf.p;
    {
      PlanHdr* h = (PlanHdr*)P->image;
      memset(h, 0, sizeof(PlanHdr));
      h->n_segs = (uint32_t)P->segs.size();
      h->total_units = P->total_units;
      h->kv_off = (uint32_t)P->kv_img_off;
      h->c2d_off = (uint32_t)P->c2d_img_off;
      h->bulk_off = (uint32_t)P->bulk_img_off;
      h->wblk_off = (uint32_t)P->wblk_img_off;
      h->n_waves = (uint32_t)P->n_waves;
      h->wave_tab_off = (uint32_t)P->wave_tab_img_off;
    }
    if (!P->segs.empty()) {
      memcpy(P->image + hdr_b, P->segs.data(), P->segs.size() * sizeof(Seg));
      memset(P->image + hdr_b + P->segs.size() * sizeof(Seg), 0, (size_t)(seg_b - (int64_t)(P->segs.size() * sizeof(Seg))));
    }
    {  // KV descriptors ordered [level 0][level 1]...[level K][staged]
      KvDesc* kvd = (KvDesc*)(P->image + P->kv_img_off);
      P->kv = kvd;
      P->n_kv = nm;
      if (nm > 0) {
        std::vector<uint32_t>& cur = W.cur;
        cur.assign(W.lvl_begin.begin(), W.lvl_begin.end() - 1);
        uint32_t scur = W.lvl_begin[K + 1];
        for (int m = 0; m < nm; ++m) {
          KvDesc d;
          d.ep_rank = mv[m].ep_rank; d.ep_page = mv[m].ep_page; d.tp_page = mv[m].tp_page;
          d.ntok_slot = (uint32_t)mv[m].ntok | (mv[m].staged ? ((uint32_t)mv[m].slot << 8) : 0u);
          if (mv[m].staged) kvd[scur++] = d; else kvd[cur[mv[m].level]++] = d;
        }
      }
      memset(P->image + P->kv_img_off + (int64_t)nm * sizeof(KvDesc), 0, (size_t)(kv_b - (int64_t)nm * (int64_t)sizeof(KvDesc)));
    }
    if (c2d_b) {
      memcpy(P->image + P->c2d_img_off, P->c2d.data(), P->c2d.size() * sizeof(C2dDesc));
      memset(P->image + P->c2d_img_off + P->c2d.size() * sizeof(C2dDesc), 0, (size_t)(c2d_b - (int64_t)(P->c2d.size() * sizeof(C2dDesc))));
    }
    if (bulk_b) {
      memcpy(P->image + P->bulk_img_off, P->bulk.data(), P->bulk.size() * sizeof(BulkDesc));
      memset(P->image + P->bulk_img_off + P->bulk.size() * sizeof(BulkDesc), 0, (size_t)(bulk_b - (int64_t)(P->bulk.size() * sizeof(BulkDesc))));
    }
    if (wblk_b) {
      memcpy(P->image + P->wblk_img_off, P->wblk.data(), P->wblk.size() * sizeof(WBlk));
      memset(P->image + P->wblk_img_off + P->wblk.size() * sizeof(WBlk), 0, (size_t)(wblk_b - (int64_t)(P->wblk.size() * sizeof(WBlk))));
    }
    {  // per wave: a header + that wave's segments with their own unit numbering and no dependencies;
       // descriptor offsets are relative to the wave's header (negative: the arrays sit before it)
      P->wave_hdr_off.assign((size_t)P->n_waves, 0);
      P->wave_units.assign((size_t)P->n_waves, 0);
      int64_t at = P->wave_img_off;
      for (int32_t w = 0; w < P->n_waves; ++w) {
        PlanHdr* h = (PlanHdr*)(P->image + at);
        memset(h, 0, sizeof(PlanHdr));
        P->wave_hdr_off[(size_t)w] = at;
        Seg* out_segs = (Seg*)(P->image + at + hdr_b);
        uint32_t n = 0, units = 0;
        bool tma = false;
        for (size_t i = 0; i < P->segs.size(); ++i) {
          if (seg_wave[i] != w) continue;
          Seg t = P->segs[i];
          t.wait_ctr = -1; t.signal_ctr = -1;
          t.unit_begin = units;
          units += t.n_units;
          tma |= seg_path(t) == PATH_TMA;
          out_segs[n++] = t;
        }
        h->n_segs = n;
        h->total_units = units;
        h->kv_off = (uint32_t)(int32_t)(P->kv_img_off - at);
        h->c2d_off = (uint32_t)(int32_t)(P->c2d_img_off - at);
        h->bulk_off = (uint32_t)(int32_t)(P->bulk_img_off - at);
        h->wblk_off = (uint32_t)(int32_t)(P->wblk_img_off - at);
        P->wave_units[(size_t)w] = units;
        at += hdr_b + (int64_t)n * (int64_t)sizeof(Seg);
      }
      uint32_t* tab = (uint32_t*)(P->image + P->wave_tab_img_off);
      memset(tab, 0, (size_t)align_up((int64_t)P->n_waves * 4, 256));
      for (int32_t w = 0; w < P->n_waves; ++w) tab[w] = (uint32_t)P->wave_hdr_off[(size_t)w];
    }
    P->tbl_image = (int32_t*)(P->image + align_up(P->image_bytes, 256));
    int32_t* T = P->tbl_image;
    memset(T, 0, kTblHdrInts * 4);
    T[0] = to; T[1] = n_req; T[2] = c.max_requests; T[3] = MP;
    for (int i = 0; i < c.max_requests; ++i) { T[kTblHdrInts + i] = -1; T[kTblHdrInts + c.max_requests + i] = 0; }
    for (int i = 0; i < n_req; ++i) { T[kTblHdrInts + i] = owner[i]; T[kTblHdrInts + c.max_requests + i] = seq_lens[i]; }
    {
      int32_t* tb = T + kTblHdrInts + 2 * c.max_requests;
      for (int i = 0; i < n_req; ++i) {
        int32_t* row = tb + (size_t)i * MP;
        memcpy(row, bt.data() + (size_t)i * MP, (size_t)npages[i] * 4);
        for (int b = npages[i]; b < MP; ++b) row[b] = -1;
      }
      P->bt = tb;
    }
    return MOEBIUS_OK;
  }

  // statistics
  int finish_stats() {
    P->stats.n_segments = (int32_t)P->segs.size();
    P->stats.n_kv_moves = nm;
    P->stats.n_kv_rounds = nm ? K + 1 + (n_staged ? 1 : 0) : 0;
    P->stats.n_kv_staged = n_staged;
    P->stats.n_pool_groups = n_pool_groups;
    P->stats.n_units = (int64_t)ub;
    P->stats.staging_used_bytes = (int64_t)n_staged * x->ep_page_bytes * (n_staged ? pools_per_group : 0);
    P->stats.desc_upload_bytes = P->image_bytes;
    P->stats.table_upload_bytes = P->tbl_bytes;
    return MOEBIUS_OK;
  }
};

}  // namespace

extern "C" int moebius_plan(moebius_ctx_t* x, moebius_mode_t from, moebius_mode_t to, int32_t n_req,
                            const int32_t* seq_lens, const int32_t* src_owner, const int32_t* src_bt,
                            moebius_plan_t** out) {
  if (!x || !out) return MOEBIUS_E_INVAL;
  *out = nullptr;
  const moebius_config_t& c = x->cfg;
  if (!((from == MOEBIUS_TP && to == MOEBIUS_EP) || (from == MOEBIUS_EP && to == MOEBIUS_TP))) return MOEBIUS_E_INVAL;
  if (n_req < 0 || n_req > c.max_requests) return MOEBIUS_E_INVAL;
  if (n_req > 0 && (!seq_lens || !src_bt)) return MOEBIUS_E_INVAL;
  if (n_req > 0 && from == MOEBIUS_EP && !src_owner) return MOEBIUS_E_INVAL;
  PlanBuilder b(x, from, to, n_req, seq_lens, src_owner, src_bt);
  int rc;
  if ((rc = b.request_state()) || (rc = b.kv_moves()) || (rc = b.kv_schedule())) return rc;   // nothing allocated yet
  if ((rc = b.new_plan())) return rc;
  if ((rc = b.weight_chain()) || (rc = b.scale_copies()) || (rc = b.attention_copies()) || (rc = b.kv_segments()) || (rc = b.merge_and_waves()) ||
      (rc = b.build_images()) || (rc = b.finish_stats()))
    return rc;                                          // the failing stage has destroyed the plan
  *out = b.P;
  return MOEBIUS_OK;
}

extern "C" int moebius_block_tables(const moebius_plan_t* p, int32_t* dst_owner, int32_t* dst_bt) {
  if (!p) return MOEBIUS_E_INVAL;
  if (dst_owner && p->n_req) memcpy(dst_owner, p->owner.data(), (size_t)p->n_req * 4);
  if (dst_bt && p->n_req)
    memcpy(dst_bt, p->bt, (size_t)p->n_req * (size_t)p->ctx->cfg.max_pages_per_request * 4);
  return MOEBIUS_OK;
}

extern "C" int moebius_plan_stats(const moebius_plan_t* p, moebius_stats_t* o) {
  if (!p || !o || o->struct_size != sizeof(moebius_stats_t)) return MOEBIUS_E_INVAL;
  *o = p->stats;
  return MOEBIUS_OK;
}

extern "C" int moebius_plan_export(const moebius_plan_t* p, int what, void* buf, int64_t cap, int64_t* needed) {
  if (!p || !needed) return MOEBIUS_E_INVAL;
  const void* src; int64_t n;
  switch (what) {
    case 0: src = p->segs.data(); n = (int64_t)p->segs.size() * sizeof(Seg); break;
    case 1: src = p->kv;          n = p->n_kv * (int64_t)sizeof(KvDesc); break;
    case 2: src = p->c2d.data();  n = (int64_t)p->c2d.size() * sizeof(C2dDesc); break;
    case 3: src = p->seg_wave.data(); n = (int64_t)p->seg_wave.size() * 4; break;
    case 4: src = p->bulk.data(); n = (int64_t)p->bulk.size() * sizeof(BulkDesc); break;
    case 5: src = p->wblk.data(); n = (int64_t)p->wblk.size() * sizeof(WBlk); break;
    default: return MOEBIUS_E_INVAL;
  }
  *needed = n;
  if (buf && cap >= n && n) memcpy(buf, src, (size_t)n);
  return MOEBIUS_OK;
}

// What the ranks [rank_lo, rank_hi) execute of a plan (wave < 0: all waves): units, bytes read, bytes
// written, and the bytes that cross between ranks (EP->TP: stored into another rank's region;
// TP->EP: loaded from another rank's region) -- the per-GPU interconnect volume of PAPER.md:189.
extern "C" int moebius_share_stats(const moebius_plan_t* P, int rank_lo, int rank_hi, int wave, int64_t* out4) {
  if (!P || !out4) return MOEBIUS_E_INVAL;
  const moebius_ctx* x = P->ctx;
  if (rank_lo < 0 || rank_hi > x->cfg.R || rank_lo >= rank_hi || wave >= P->n_waves) return MOEBIUS_E_INVAL;
  DevParams p;
  memset(&p, 0, sizeof(p));
  p.kv = P->kv;
  p.c2d = P->c2d.data();
  p.bulk = P->bulk.data();
  p.wblk = P->wblk.data();
  p.rank_stride = x->rank_stride;
  int64_t units = 0, rd = 0, wr = 0, cross = 0;
  for (size_t si = 0; si < P->segs.size(); ++si) {
    if (wave >= 0 && P->seg_wave[si] != wave) continue;
    const Seg& s = P->segs[si];
    for (uint32_t u = 0; u < s.n_units; ++u) {
      const int q = (int)unit_ep_rank(s, p, u);
      if (q < rank_lo || q >= rank_hi) continue;
      ++units;
      if (seg_kind(s) == SEG_COPY2D) {
        const C2dDesc& d = p.c2d[s.desc_begin + u];
        const int64_t b = (int64_t)d.rows * d.run_bytes;
        rd += b; wr += b;
        if (d.src_off / x->rank_stride != d.dst_off / x->rank_stride) cross += b;
        continue;
      }
      if (seg_kind(s) == SEG_BULK) {
        BulkUnit bu;
        decode_bulk(s, p, u, bu);
        const int64_t b = (int64_t)bu.nrows * bu.piece;
        rd += b; wr += b;
        if (!(s.kv_mode & 3u)) cross += b;     // attention gather: always from another rank's shard; a parked
        continue;                               // block stays on its rank
      }
      if (seg_kind(s) == SEG_XPOSE) {
        Box bx;
        decode_box(s, p, u, 0, bx);
        const int64_t per_group = (int64_t)bx.nrows * s.chunk_bytes;
        rd += per_group * s.groups_per_unit; wr += per_group * s.groups_per_unit;
        // a block moving between the EP rows and its staging slot stays on its rank (kv_mode & 1: the EP
        // side is the slot, so only the TP pieces of other ranks cross)
        for (uint32_t g = bx.g0; g < bx.g0 + s.groups_per_unit; ++g)
          if ((int)g != q) cross += per_group;
        continue;
      }
      uint32_t pb, di;
      kv_unit(s, u, pb, di);
      const KvDesc& d = p.kv[s.desc_begin + di];
      const int64_t row = (int64_t)(d.ntok_slot & 0xFFu) * s.run_bytes * seg_boxes(s, u);   // one group, all pools of the unit
      if (s.kv_mode == KV_STG_COPY) { rd += row * s.n_groups; wr += row * s.n_groups; continue; }
      rd += row * s.n_groups;
      if (s.ep_is_src) {
        wr += row * s.n_groups * s.rep;
        cross += row * ((int64_t)s.n_groups * s.rep - 1);
      } else {
        wr += row * s.n_groups;
        for (uint32_t g = 0; g < s.n_groups; ++g)
          if ((int)tp_src_rank(g, s.rep, d.ep_rank) != d.ep_rank) cross += row;
      }
    }
  }
  out4[0] = units; out4[1] = rd; out4[2] = wr; out4[3] = cross;
  return MOEBIUS_OK;
}
