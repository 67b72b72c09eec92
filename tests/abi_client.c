/* A plain C99 client of the C ABI (host-only calls): proves that include/moebius.h + libmoebius.so
 * are usable without Python, torch or C++.  Built and run by tests/test_abi.py.  BASELINE.json
 * config 1 shapes; the expected byte count is the closed form (1 - 1/R) * L * 3 * E * H * I * b. */
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "moebius.h"

#define CHECK(x) do { int rc_ = (x); if (rc_ != MOEBIUS_OK) { printf("FAIL %s -> %s\n", #x, moebius_status_str(rc_)); return 1; } } while (0)

int main(void) {
  moebius_config_t c;
  memset(&c, 0, sizeof(c));
  c.struct_size = sizeof(c);
  c.R = 2; c.L = 1; c.E = 8; c.H = 64; c.I = 32;
  c.w_dtype = MOEBIUS_BF16; c.w_orient = 0;
  c.kv_heads = 2; c.head_dim = 16; c.page_tokens = 16; c.kv_dtype = MOEBIUS_BF16;
  c.kv_pool_bytes_per_rank_layer = 16 * 2 * 16 * 2 * 64;   /* 64 EP pages */
  c.max_requests = 4; c.max_pages_per_request = 4;
  c.staging_cap_bytes = 0;
  moebius_ctx_t* ctx = NULL;
  CHECK(moebius_create(&c, &ctx));
  moebius_layout_t lay;
  memset(&lay, 0, sizeof(lay));
  lay.struct_size = sizeof(lay);
  CHECK(moebius_layout(ctx, &lay));
  if (lay.pages_ep != 64 || lay.pages_tp != 128 || lay.base_bytes != 2 * lay.rank_stride_bytes) { printf("FAIL layout\n"); return 1; }
  moebius_view_t v;
  memset(&v, 0, sizeof(v));
  v.struct_size = sizeof(v);
  CHECK(moebius_view(ctx, MOEBIUS_TP, 1, 0, MOEBIUS_T_GATE, &v));
  if (v.shape[0] != 8 || v.shape[1] != 64 || v.shape[2] != 16 || v.offset < lay.rank_stride_bytes) { printf("FAIL view\n"); return 1; }

  int32_t lens[4] = {5, 16, 17, 64};
  int32_t bt[4][4] = {{0, -1, -1, -1}, {1, -1, -1, -1}, {2, 3, -1, -1}, {4, 5, 6, 7}};
  moebius_plan_t* plan = NULL;
  CHECK(moebius_plan(ctx, MOEBIUS_TP, MOEBIUS_EP, 4, lens, NULL, &bt[0][0], &plan));
  moebius_stats_t st;
  memset(&st, 0, sizeof(st));
  st.struct_size = sizeof(st);
  CHECK(moebius_plan_stats(plan, &st));
  if (st.w_moved != 49152 || st.n_kv_moves != 8) { printf("FAIL stats %lld %d\n", (long long)st.w_moved, st.n_kv_moves); return 1; }
  int32_t owner[4], nbt[4][4];
  CHECK(moebius_block_tables(plan, owner, &nbt[0][0]));
  /* longest first onto the least loaded rank: 64 -> r0, 17 -> r1, 16 -> r1, 5 -> r1 */
  if (owner[3] != 0 || owner[2] != 1 || owner[1] != 1 || owner[0] != 1) { printf("FAIL partition\n"); return 1; }
  if (nbt[3][0] != 63 || nbt[3][3] != 60 || nbt[0][0] != 63 || nbt[0][1] != -1) { printf("FAIL tables\n"); return 1; }
  int32_t n_waves = 0;
  CHECK(moebius_plan_waves(plan, &n_waves));
  int64_t share[4];
  CHECK(moebius_share_stats(plan, 0, 2, -1, share));
  if (n_waves != 3 || share[3] != st.w_moved + st.kv_moved) { printf("FAIL waves/share\n"); return 1; }
  /* no device on this path: the execution entry point refuses instead of falling back */
  if (moebius_reshard(ctx, plan, NULL) != MOEBIUS_E_STATE) { printf("FAIL reshard without bind\n"); return 1; }
  moebius_plan_destroy(plan);

  moebius_policy_config_t pc;
  memset(&pc, 0, sizeof(pc));
  pc.struct_size = sizeof(pc);
  CHECK(moebius_policy_preset(MOEBIUS_POLICY_INTERACTIVE, 256.0, 5.0, &pc));
  moebius_policy_t* pol = NULL;
  CHECK(moebius_policy_create(&pc, MOEBIUS_TP, &pol));
  int32_t dec = -1, mode = -1;
  CHECK(moebius_policy_step(pol, NULL, 0.0, 300, NULL, &dec, &mode));
  if (dec != MOEBIUS_DECISION_SWITCH || mode != MOEBIUS_EP || pc.W != 8) { printf("FAIL policy\n"); return 1; }
  moebius_policy_destroy(pol);
  moebius_destroy(ctx);
  printf("OK version %d\n", moebius_version());
  return 0;
}
