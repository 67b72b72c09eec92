// moebius_host.h -- host-side objects behind the opaque C handles (product code, not the oracle).
#ifndef MOEBIUS_HOST_H_
#define MOEBIUS_HOST_H_

#include <cstdint>
#include <vector>

#include "../../include/moebius.h"
#include "moebius_units.h"

namespace moebius {

constexpr int kMaxCounters = 16384;
constexpr int kMaxSegs = 32768;
constexpr int64_t kHdrBytes = 256;                         // ticket lives at byte 0
constexpr int64_t kCtrOff = kHdrBytes;                     // uint32 counters[kMaxCounters]
constexpr int64_t kSegOff = kCtrOff + 4 * kMaxCounters;    // Seg[...]
constexpr int kTblHdrInts = 16;
constexpr int kTimingRing = 64;

struct ImageBuf {            // host upload image of a plan; pinned when a CUDA device is present
  char* p;
  int64_t bytes;
  bool pinned;
  void* ev;                  // cudaEvent_t recorded after the last upload that reads this buffer (or null)
};

struct Move {                // one live (request, block) page under both modes
  int32_t req, blk, ep_rank, ep_page, tp_page, ntok;
  int32_t level;
  int32_t slot;
  uint8_t staged;
};

// Planner workspace, kept by the context so that a steady stream of switches re-uses warm memory
// (a fresh multi-megabyte vector per plan costs more in page faults than the planning itself).
struct PlanScratch {
  std::vector<int32_t> npages, order, owner, bt, reader, indeg, queue, stamp;
  std::vector<int32_t> blk_off, blk, dep_off, dep, dep_cur;   // CSR: blockers of m, dependents of b
  std::vector<int64_t> tok, cnt, used;
  std::vector<uint8_t> seen, done, self_staged;
  std::vector<uint32_t> lvl_begin, cur;
  std::vector<Move> mv;
};

// One expert-weight object of a layer = one link of the slot chain (PAPER.md:150-156 at (layer,
// matrix) grain).  Its EP view of rank q is [rows][R runs][run bytes], its TP view of rank j is
// [q][rows][run bytes].  Offsets in units of the slot size S.
struct WObj {
  int tensor_id;             // moebius_tensor_t of the weight; scale tensor id in scale_id
  int scale_id;
  int slot, n_slots;         // TP view starts at slot `slot` of the layer's 3 slots; size n_slots * S
  int long_run;              // 0: run = (I/R)*b, rows = (E/R)*H (the intermediate axis is last)
                             // 1: run = (I/R)*H*b, rows = (E/R)*row_mult (the intermediate axis is in the middle)
  int row_mult;              // 2 for the stacked W13 (gate block, up block), else 1
};

struct ScaleGeom {           // fp8 block scales of one matrix kind (reading A13)
  int64_t tp_bytes;          // per rank, allocated with the largest nb over ranks
  int64_t ep_bytes;          // per rank
};

}  // namespace moebius

struct moebius_ctx {
  moebius_config_t cfg;
  int wb, kvb;                    // element bytes
  int ep_shift;                   // the EP view of an object starts ep_shift slots after its TP view
                                  // (= the largest object, in slots; 0 when R == 1)
  int n_obj;                      // objects per layer: 3 (gate, up, down) or 2 (W13, W2)
  moebius::WObj obj[3];
  int64_t S;                      // weight slot bytes per rank
  int64_t w_off, scale_tp_off, scale_ep_off, kv_off, rank_stride;
  int64_t flag_off;               // per rank region: the round-barrier flag page, uint32 flag[kMaxCounters]
  moebius::ScaleGeom sg[3];
  int64_t scale_tp_layer, scale_ep_layer;  // bytes per layer per rank
  // attention projections (attn_mode != 0): per rank and layer the four full tensors,
  // then (MOEBIUS_ATTN_DUAL) the four head shards; offsets within one layer's block
  int64_t attn_off, attn_layer_bytes, attn_full_off[4], attn_shard_off[4], attn_full_sz[4], attn_shard_sz[4];
  int64_t attn_full_bytes, attn_dup_bytes;   // all ranks and layers
  int64_t max_bulk;
  int G, rep, hpr;
  int64_t run_kv, ep_page_bytes, tp_page_bytes, pool_bytes;
  int32_t pages_ep, pages_tp;
  int64_t staging_bytes, desc_bytes, table_bytes, resident_bytes, spare_bytes;
  int64_t w_stg_bytes;            // tail of the staging buffer reserved for parked weight blocks (S2); 0 when every
                                  // object moves out of place
  int64_t max_wblk;
  int64_t max_kv_desc, max_c2d;
  // bound buffers
  bool bound;
  char* base;
  char* stg;
  char* desc;
  int32_t* tables;
  int active_mode;
  int64_t switch_count;
  // launch shape (PATH_LSU tuning) and the TMA path's geometry (fixed before the first plan)
  int ctas_per_sm, threads, unit_kb;
  int chain_bands;                // 1 (default): equal-sized objects are chained half by half (no drain between links)
  int kv_slice_floor;             // smallest KV slice the merge interleaves with the weight chain, in units (0: default)
  int kv_max_level;               // longest chain of dependent KV rounds before chains are cut by staging
  int use_tma;                    // planner emits PATH_TMA segments where the shapes allow
  int n_pipes;                    // TMA pipes (warps) per CTA, one CTA per SM
  int64_t stage_bytes;            // largest PATH_TMA unit (what the planner sizes units to)
  int64_t ring_bytes;             // shared-memory ring of one pipe (units take what they need, FIFO)
  int ld_max;                     // units of one pipe whose loads may be in flight at once
  int l2_ld, l2_st;               // L2 cache-hint policy of the TMA loads / stores (0: none)
  int def_pipes;                  // the defaults moebius_create derived from the EP page size
  int64_t def_stage_bytes;
  int xt_ok, kt_ok;               // weight / KV tensor maps exist for this config
  int xt_rows;                    // rows of the weight tensor-map box
  int kt_pools;                   // pools per KV unit
  alignas(64) unsigned char tmap_w[128];   // CUtensorMap storage (encoded at bind time)
  alignas(64) unsigned char tmap_kv[128];
  alignas(64) unsigned char tmap_wtp[128];  // the TP views of the weight slots (xt_mode 1)
  int xt_mode;                    // 1 (default): weight boxes over the TP views; 0: over the EP views
  int xt_promo;                   // L2 promotion of that tensor map (0 none, 1/2/3 = 64/128/256 B; tuning)
  alignas(64) unsigned char tmap_stg[128];  // the staging buffer as an array of EP-page images
  bool tmaps_valid;
  bool prepared;                  // device_prepare has run for the current buffers and stage geometry
  size_t smem_set;                // dynamic shared memory the kernel attribute is currently set to
  // device facts + timing (filled lazily by the CUDA side)
  int n_sm;
  int timing;
  void* ev[2 * moebius::kTimingRing];   // event pairs (begin, end) round the kernel, a ring
  int64_t ev_count;                     // pairs recorded so far
  bool ev_valid;
  // upload images released by destroyed plans, reused by the next moebius_plan (pinning a fresh
  // buffer costs milliseconds; a switch must not pay it every time)
  std::vector<moebius::ImageBuf> image_pool;
  moebius::PlanScratch scratch;
  int has_device;                       // -1 unknown, 0 no CUDA device (host-only planner), 1 yes
  char* mailbox;                        // pinned, fixed address: [work-list image capacity][tables]; what
                                        // moebius_reshard_staged uploads (allocated by the first moebius_stage_plan)
};

struct moebius_plan {
  moebius_ctx* ctx;
  int from, to, n_req;
  std::vector<moebius::Seg> segs;
  std::vector<moebius::C2dDesc> c2d;
  std::vector<moebius::BulkDesc> bulk;
  std::vector<moebius::WBlk> wblk;
  const moebius::KvDesc* kv;      // n_kv descriptors, inside `image`
  int64_t n_kv;
  std::vector<int32_t> lens, owner;   // target-mode request state
  const int32_t* bt;              // [n_req][max_pages_per_request], inside `tbl_image`
  moebius_stats_t stats;
  uint32_t n_counters, total_units;
  bool uses_tma;                  // some segment is PATH_TMA: needs the pipes' shared-memory rings
  int64_t stage_bytes; int xt_rows;   // geometry the plan was built for
  // one contiguous upload image: [segs][kv][c2d], and the table image; pinned when CUDA allows
  char* image;
  int64_t image_bytes, kv_img_off, c2d_img_off, bulk_img_off, wblk_img_off, wave_tab_img_off;
  // rank-share execution (multi-GPU): per dependency wave a header + segment list inside the image
  int32_t n_waves;
  int64_t wave_img_off;
  std::vector<int32_t> seg_wave;       // dependency wave of every segment
  std::vector<int64_t> wave_hdr_off;
  std::vector<uint32_t> wave_units;
  int32_t* tbl_image;
  int64_t tbl_bytes;
  moebius::ImageBuf buf;          // backing storage of image + tbl_image
};

namespace moebius {
// CUDA side (moebius_cuda.cu)
bool image_acquire(moebius_ctx* ctx, int64_t bytes, ImageBuf* out);   // from the pool, else fresh
void image_release(moebius_ctx* ctx, const ImageBuf& buf);             // back to the pool (bounded)
void image_free(const ImageBuf& buf);
void cuda_ctx_destroy(moebius_ctx* ctx);
void lpt_partition(int n_req, const int32_t* seq_lens, int R, PlanScratch& scratch, int32_t* owner);
int device_prepare(moebius_ctx* ctx);  // one-off device-side setup of a bound context (moebius_bind, moebius_set_tma)
void tma_geometry(moebius_ctx* ctx);   // derives xt_ok/kt_ok/xt_rows/kt_pools from cfg + stage_bytes (host only)
}  // namespace moebius

#endif
