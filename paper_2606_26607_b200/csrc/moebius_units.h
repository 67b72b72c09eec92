// moebius_units.h -- work-list format and unit decode, shared by the host planner and the sm_100a
// kernel (both are the product; the CPU oracle under oracle/ shares nothing with this file).
//
// A plan is an ordered list of SEGMENTS; a segment is n_units independent work UNITS of one kind;
// a unit is what one warp executes.  Units are handed out in list order by one global ticket.
// A segment may WAIT on a completion counter (all units that signal that counter have finished)
// and may SIGNAL one.  Dependencies always point backwards in list order, so in-order hand-out is
// deadlock-free whatever the number of resident warps.
//
// Every data move is one of three shapes:
//   XBOX  "run transposition": an EP-side block [rows][J runs][cc*16 B] that is contiguous per row,
//         against J TP-side blocks [rows][cc*16 B], one per group (each on `rep` ranks).  This is
//         the paper's owner-changed slice: expert weights (rank q's EP row holds
//         the R TP shards of that row side by side) and KV pages (an EP page row
//         = one token's G head groups side by side; a TP page row = one group).
//   LIN   contiguous copy (KV page <-> staging slot).
//   C2D   small 2-D strided copy in 4-byte elements (fp8 block scales).
//   BULK  large 2-D strided copy in 16-byte elements: n_desc descriptors of one shape (rows x run with a
//         source and a destination row stride), split into units of whole rows or of run chunks
//         (attention head shards gathered TP->EP).
#ifndef MOEBIUS_UNITS_H_
#define MOEBIUS_UNITS_H_

#include <stdint.h>

#if defined(__CUDACC__)
#define MB_HD __host__ __device__ __forceinline__
#else
#define MB_HD inline
#endif

namespace moebius {

enum : uint32_t { SEG_XPOSE = 0, SEG_KV = 1, SEG_COPY2D = 2, SEG_BULK = 3 };
enum : uint32_t { KV_MOVE = 0, KV_MOVE_STG = 1, KV_STG_COPY = 2 };
// How the kernel executes a segment's units (bits 8..15 of Seg::kind).  The unit geometry is the
// same for both paths (decode_box below is the single definition); only the data path differs:
//   PATH_LSU  one warp copies the unit with 16-byte ld.global / st.global
//   PATH_TMA  one elected lane moves it through a shared-memory stage with TMA: the EP side is ONE
//             cp.async.bulk.tensor over a 5-D tensor map whose box is the whole unit (the run
//             transposition happens in the box: smem holds [group][row][run]), the TP side is one
//             contiguous cp.async.bulk per (group, replica).  Units with a single group (chunks of
//             long runs, e.g. the down projection) use plain 1-D bulk copies on both sides.  Staged KV
//             pages use a second tensor map over the staging buffer (an array of page images).
enum : uint32_t { PATH_LSU = 0, PATH_TMA = 1 };

struct Seg {              // 128 bytes, uploaded verbatim
  uint32_t kind;          // bits 0..7: SEG_*; bits 8..15: PATH_*
  uint32_t ep_is_src;     // 1: EP side is read, TP side written (EP->TP); 0: the reverse
  int32_t  wait_ctr;      // -1: none
  uint32_t wait_target;
  int32_t  signal_ctr;    // -1: none
  uint32_t unit_begin;    // global id of this segment's first unit
  uint32_t n_units;
  uint32_t run_bytes;     // one group's contiguous piece of an EP row (= TP row)
  uint32_t n_groups;      // runs per EP row: R (weights) or G = min(kv_heads, R) (KV)
  uint32_t rep;           // TP ranks per group: 1 (weights) or max(1, R/kv_heads) (KV)
  uint32_t rows_per_unit;
  uint32_t groups_per_unit;  // n_groups, or 1 when a run is split into chunks
  uint32_t chunk_bytes;      // bytes of a run one unit handles (== run_bytes unless chunked)
  uint32_t chunks_per_run;
  uint32_t rows_total;       // XPOSE: rows per EP rank (E/R*H for gate/up, E/R for down)
  uint32_t row_blocks;       // XPOSE: ceil(rows_total / rows_per_unit)
  int64_t  ep_off;           // XPOSE: EP view offset in the rank region; KV: pool 0 offset; BULK: source row stride
  int64_t  tp_off;           // XPOSE: TP view offset in the rank region; KV: == ep_off;   BULK: destination row stride
  uint32_t kv_mode;
  uint32_t desc_begin;       // first descriptor (KV move or C2D) of this segment; XPOSE: EP slot index
  uint32_t n_desc;
  uint32_t pool_begin;       // KV: first pool (z = 2*layer + {K:0,V:1}) of this segment
  uint32_t n_pools;
  uint32_t pools_per_unit;
  uint32_t ep_page_bytes;
  uint32_t tp_page_bytes;
  int64_t  pool_bytes;
  uint32_t stg_pool_begin;   // KV staging: slot s, pool z lives at ((s*stg_pools)+(z-stg_pool_begin))*ep_page_bytes
  uint32_t stg_pools;
};
static_assert(sizeof(Seg) == 128, "Seg must be 128 bytes");

struct KvDesc {           // 16 bytes: one (request, block) page move, layer- and K/V-agnostic
  int32_t  ep_rank;       // EP-side owner of the request (one index vector for all layers)
  int32_t  ep_page;       // EP page id in that rank's pool
  int32_t  tp_page;       // TP page id (same on every rank)
  uint32_t ntok_slot;     // bits 0..7: valid tokens in the page (1..page_tokens <= 255);
                          // bits 8..31: staging slot (KV_MOVE_STG / KV_STG_COPY segments only)
};
static_assert(sizeof(KvDesc) == 16, "KvDesc must be 16 bytes");

struct C2dDesc {          // 32 bytes: rows x run_bytes, 4-byte elements, offsets from dev_base
  int64_t  src_off, dst_off;
  uint32_t rows, run_bytes, src_stride, dst_stride;
};
static_assert(sizeof(C2dDesc) == 32, "C2dDesc must be 32 bytes");

// XPOSE block-list mode (an object whose EP view overlaps its own TP view is moved
// block by block in dependency waves, blocks on cycles parked in the bounded staging buffer).  A block is
// rows [row0, row0 + nrows) of EP rank q; `slot` is its staging slot when the segment's EP side is the
// staging buffer (Seg::kv_mode & 1).  Fields reused by such a segment: n_desc = number of blocks (0 = the
// whole object, the common case), pool_begin = first WBlk, pools_per_unit = units per block, pool_bytes =
// bytes of one staging slot.  REGULAR block lists (the banded chain: the same rows of consecutive ranks)
// carry no descriptors at all -- a dependent global load per unit costs the issuing pipe a tenth of its
// rate: stg_pools = 1 marks them, block i is rows [pool_begin, pool_begin + n_pools) of rank stg_pool_begin + i.
struct WBlk {
  uint32_t q, row0, nrows, slot;
};
static_assert(sizeof(WBlk) == 16, "WBlk must be 16 bytes");

struct BulkDesc {         // 16 bytes: one strided copy of the segment's shape; offsets from dev_base, or from
                          // the weight part of the staging buffer when Seg::kv_mode has bit 0 (source) /
                          // bit 1 (destination) set
  int64_t  src_off, dst_off;
};
static_assert(sizeof(BulkDesc) == 16, "BulkDesc must be 16 bytes");

// First 256 bytes of the uploaded work-list image.  Everything that differs from plan to plan is
// read by the kernel from here, so the kernel's ARGUMENTS are the same for every switch of a
// context and the launch can sit in a captured CUDA graph (moebius_reshard_staged).
struct PlanHdr {
  uint32_t n_segs;
  uint32_t total_units;
  uint32_t kv_off;        // byte offsets from the start of the image
  uint32_t c2d_off;
  uint32_t bulk_off;
  uint32_t wblk_off;
  uint32_t n_waves;       // main header only: dependency waves, and where their headers are (wave_tab_off:
  uint32_t wave_tab_off;  // uint32[n_waves], byte offsets of the per-wave headers from the start of the image)
  uint32_t pad_[56];
};
static_assert(sizeof(PlanHdr) == 256, "PlanHdr must be 256 bytes");

struct DevParams {        // decoded launch state (the kernel fills the plan-dependent fields from PlanHdr)
  char*            base;
  char*            stg;
  const PlanHdr*   hdr;           // the uploaded image; segs/kv/c2d/n_segs/total_units below come from it
  const Seg*       segs;
  const KvDesc* kv;
  const C2dDesc*   c2d;
  const BulkDesc*  bulk;
  const WBlk*      wblk;
  int64_t          wstg_off;      // weight part of the staging buffer (its tail), bytes from `stg`
  uint32_t*        ticket;
  uint32_t*        counters;
  int64_t          rank_stride;
  uint32_t         n_segs;
  uint32_t         total_units;
  uint32_t         stage_bytes;   // PATH_TMA: largest unit (the planner's unit size)
  uint32_t         ring_bytes;    // PATH_TMA: bytes of one pipe's shared-memory ring (>= stage_bytes)
  uint32_t         ld_max;        // PATH_TMA: units of one pipe whose loads may be in flight at once
  uint32_t         l2_ld, l2_st;  // PATH_TMA: L2 cache-hint policy of loads / stores (0 none, 1 evict_first, 2 evict_last, ...)
  uint32_t         xt_rows;       // PATH_TMA: rows of the weight tensor-map box (= rows_per_unit)
  uint32_t         page_tokens;
  uint32_t         n_ranks;       // R
  uint32_t         rank_lo, rank_hi;   // rank share: only units whose EP-side rank is in [lo, hi) are
                                       // executed (multi-GPU: the ranks this GPU owns); [0, R) = all
  // Device-side round barrier (one cross-GPU barrier per dependency round).
  // n_shares > 0: this launch executes shares [share_first, share_first + share_count) of n_shares --
  // its CTAs are split evenly among them -- wave by wave; share s owns ranks [share_bounds[s],
  // share_bounds[s+1]).  After a wave the last CTA of a share raises that share's flag for the wave
  // (st.release.sys) in the flag page of the share's first rank; every CTA then waits for the flags of
  // ALL n_shares shares (ld.acquire.sys) -- on several GPUs those are peer addresses.
  uint32_t         xt_mode;       // PATH_TMA weight boxes: 0 = tensor map over the EP views, 1 = over the TP views
  uint32_t         ep_shift;      // slots between a TP view and its EP view
  uint32_t         n_shares, share_first, share_count;
  int64_t          flag_off;           // flag page offset inside a rank region: uint32 flag[wave]
  uint8_t          share_bounds[72];
};

MB_HD uint32_t seg_kind(const Seg& s) { return s.kind & 0xFFu; }
MB_HD uint32_t seg_path(const Seg& s) { return (s.kind >> 8) & 0xFFu; }

// One executable shape.  lin != 0: contiguous copy of lin_bytes from src to dst.
struct Box {
  char*    ep;            // EP-side row 0 (first group / chunk of this unit)
  char*    tp;            // TP-side row 0 at rank 0; add rank*rank_stride
  uint32_t ep_row_stride, tp_row_stride;
  uint32_t nrows, J, g0, cc;   // cc = 16-byte chunks per (row, group)
  uint32_t run_bytes, rep;
  int32_t  owner;         // TP->EP source rule: group g is read from `owner` if it holds g, else
                          // from the lowest-rank holder g*rep (reading A5); -1: rank g
  uint32_t lin;
  char    *lin_src, *lin_dst;
  uint64_t lin_bytes;
  uint32_t q, row0;       // XPOSE: EP rank and first row of this unit (tensor-map coordinates)
};

// KV unit u of a segment = (pool block pb, descriptor di), pool-block-major: consecutive units are
// consecutive page descriptors of the SAME pools, so concurrently running pipes touch neighbouring
// pages (canonical tables hand out consecutive pages) instead of 2L pools x R ranks far apart.
MB_HD void kv_unit(const Seg& s, uint32_t u, uint32_t& pb, uint32_t& di) {
  pb = u / s.n_desc;
  di = u - pb * s.n_desc;
}

MB_HD uint32_t seg_boxes(const Seg& s, uint32_t u) {
  if (seg_kind(s) != SEG_KV) return 1;
  uint32_t pb, di;
  kv_unit(s, u, pb, di);
  uint32_t z0 = pb * s.pools_per_unit;
  uint32_t n = s.n_pools - z0;
  return n < s.pools_per_unit ? n : s.pools_per_unit;
}

// TP rank that holds the copy of group g that is READ in a TP->EP move.
MB_HD uint32_t tp_src_rank(uint32_t g, uint32_t rep, int32_t owner) {
  if (owner >= 0 && (uint32_t)owner / rep == g) return (uint32_t)owner;
  return g * rep;
}

// EP-side rank of a unit: the rank whose EP view it reads (EP->TP: pushed to the TP owners) or writes
// (TP->EP: pulled from the TP holders).  PAPER.md:172: "each kernel reads from the source-mode alias
// and writes the slice into the peer's target-mode slot" -- on several GPUs a unit runs on the GPU
// that owns this rank.
MB_HD uint32_t unit_ep_rank(const Seg& s, const DevParams& p, uint32_t u) {
  if (seg_kind(s) == SEG_XPOSE) {
    if (s.n_desc) return s.stg_pools ? s.stg_pool_begin + u / s.pools_per_unit : p.wblk[s.pool_begin + u / s.pools_per_unit].q;
    u /= s.chunks_per_run;
    u /= s.n_groups / s.groups_per_unit;
    return u / s.row_blocks;
  }
  if (seg_kind(s) == SEG_KV) {
    uint32_t pb, di;
    kv_unit(s, u, pb, di);
    return (uint32_t)p.kv[s.desc_begin + di].ep_rank;
  }
  if (seg_kind(s) == SEG_BULK) {    // pulled by the rank that receives it
    const uint32_t per_desc = s.row_blocks * s.chunks_per_run;
    const BulkDesc d = p.bulk[s.desc_begin + u / per_desc];
    // a copy into / out of the staging buffer belongs to the rank whose bytes it parks
    return (uint32_t)(((s.kv_mode & 2u) ? d.src_off : d.dst_off) / p.rank_stride);
  }
  const C2dDesc& d = p.c2d[s.desc_begin + u];
  return (uint32_t)((s.ep_is_src ? d.src_off : d.dst_off) / p.rank_stride);
}

// BULK unit u (local to the segment): descriptor u / (row_blocks*chunks_per_run); within it row block rb
// and run chunk ch.  The unit copies `nrows` pieces of chunk_bytes; piece t is at src + t*src_stride.
struct BulkUnit {
  char *src, *dst;
  int64_t src_stride, dst_stride;
  uint32_t nrows, piece;     // piece = bytes per row handled by this unit
};
MB_HD void decode_bulk(const Seg& s, const DevParams& p, uint32_t u, BulkUnit& b, bool has_pre = false, BulkDesc pre = BulkDesc{0, 0}) {
  const uint32_t per_desc = s.row_blocks * s.chunks_per_run;
  const uint32_t di = u / per_desc, w = u - di * per_desc;
  const uint32_t rb = w / s.chunks_per_run, ch = w - rb * s.chunks_per_run;
  const BulkDesc d = has_pre ? pre : p.bulk[s.desc_begin + di];
  const uint32_t row0 = rb * s.rows_per_unit;
  uint32_t nrows = s.rows_total - row0;
  if (nrows > s.rows_per_unit) nrows = s.rows_per_unit;
  b.nrows = nrows;
  b.piece = s.chunk_bytes;
  b.src_stride = s.ep_off;
  b.dst_stride = s.tp_off;
  char* sb = (s.kv_mode & 1u) ? p.stg + p.wstg_off : p.base;
  char* db = (s.kv_mode & 2u) ? p.stg + p.wstg_off : p.base;
  b.src = sb + d.src_off + (int64_t)row0 * s.ep_off + (int64_t)ch * s.chunk_bytes;
  b.dst = db + d.dst_off + (int64_t)row0 * s.tp_off + (int64_t)ch * s.chunk_bytes;
}

// Decode box k of unit u (u is LOCAL to the segment).
// `pre`: the unit's WBlk descriptor if the caller has fetched it already (block lists: the TMA pipes prefetch
// it with the ticket, so that no dependent global load sits between a ticket and its first TMA operation).
MB_HD void decode_box(const Seg& s, const DevParams& p, uint32_t u, uint32_t k, Box& b, bool has_pre = false, WBlk pre = WBlk{0, 0, 0, 0}) {
  b.lin = 0;
  b.run_bytes = s.run_bytes;
  b.rep = s.rep;
  b.tp_row_stride = s.run_bytes;
  if (seg_kind(s) == SEG_XPOSE) {
    const uint32_t jgroups = s.n_groups / s.groups_per_unit;
    uint32_t q, row0, row_end, blk_row0 = 0, slot = 0;
    if (s.n_desc) {                       // block-list mode: unit = (block, row block, group block, chunk)
      const uint32_t di = u / s.pools_per_unit;
      u -= di * s.pools_per_unit;
      if (s.stg_pools) {                  // regular: computed, no descriptor
        q = s.stg_pool_begin + di; blk_row0 = s.pool_begin; row_end = s.pool_begin + s.n_pools;
      } else {
        const WBlk k = has_pre ? pre : p.wblk[s.pool_begin + di];
        q = k.q; blk_row0 = k.row0; row_end = k.row0 + k.nrows; slot = k.slot;
      }
    } else {
      q = u / (s.row_blocks * jgroups * s.chunks_per_run);
      u -= q * (s.row_blocks * jgroups * s.chunks_per_run);
      row_end = s.rows_total;
    }
    const uint32_t ch = u % s.chunks_per_run;  u /= s.chunks_per_run;
    const uint32_t jg = u % jgroups;           const uint32_t rb = u / jgroups;
    row0 = blk_row0 + rb * s.rows_per_unit;
    uint32_t nrows = row_end - row0;
    if (nrows > s.rows_per_unit) nrows = s.rows_per_unit;
    b.nrows = nrows;
    b.q = q; b.row0 = row0;
    b.J = s.groups_per_unit;
    b.g0 = jg * s.groups_per_unit;
    b.cc = s.chunk_bytes >> 4;
    b.owner = -1;
    b.ep_row_stride = s.n_groups * s.run_bytes;
    int64_t tp = s.tp_off + ((int64_t)q * s.rows_total + row0) * s.run_bytes + (int64_t)ch * s.chunk_bytes;
    b.tp = p.base + tp;
    if (s.n_desc && (s.kv_mode & 1u)) {   // the block's EP rows live in its staging slot
      b.ep = p.stg + p.wstg_off + (int64_t)slot * s.pool_bytes +
             ((int64_t)(row0 - blk_row0) * s.n_groups + b.g0) * s.run_bytes + (int64_t)ch * s.chunk_bytes;
    } else {
      b.ep = p.base + (int64_t)q * p.rank_stride + s.ep_off +
             ((int64_t)row0 * s.n_groups + b.g0) * s.run_bytes + (int64_t)ch * s.chunk_bytes;
    }
    return;
  }
  // SEG_KV
  uint32_t pb, di;
  kv_unit(s, u, pb, di);
  uint32_t z = s.pool_begin + pb * s.pools_per_unit + k;
  KvDesc d = p.kv[s.desc_begin + di];
  uint32_t ntok = d.ntok_slot & 0xFFu;
  uint32_t slot = d.ntok_slot >> 8;
  int64_t pool = s.ep_off + (int64_t)z * s.pool_bytes;
  char* ep_pool = p.base + (int64_t)d.ep_rank * p.rank_stride + pool + (int64_t)d.ep_page * s.ep_page_bytes;
  char* ep_stg = p.stg + ((int64_t)slot * s.stg_pools + (z - s.stg_pool_begin)) * (int64_t)s.ep_page_bytes;
  uint32_t row_bytes = s.n_groups * s.run_bytes;
  if (s.kv_mode == KV_STG_COPY) {
    b.lin = 1;
    b.lin_bytes = (uint64_t)ntok * row_bytes;
    // ep_is_src: the pool page is saved into its staging slot; else the slot is written back
    b.lin_src = s.ep_is_src ? ep_pool : ep_stg;
    b.lin_dst = s.ep_is_src ? ep_stg : ep_pool;
    return;
  }
  b.ep = (s.kv_mode == KV_MOVE_STG) ? ep_stg : ep_pool;
  b.tp = p.base + pool + (int64_t)d.tp_page * s.tp_page_bytes;
  b.ep_row_stride = row_bytes;
  b.nrows = ntok;
  b.J = s.n_groups;
  b.g0 = 0;
  b.cc = s.run_bytes >> 4;
  b.owner = d.ep_rank;
}

// Addresses of 16-byte chunk idx of a box (idx < nrows*J*cc, EP-side linear order).
// tp_rel excludes the rank term; the caller adds rank*rank_stride.
MB_HD void box_chunk(const Box& b, uint32_t idx, char*& ep, char*& tp_rel, uint32_t& group) {
  uint32_t per_row = b.J * b.cc;
  uint32_t t = idx / per_row;
  uint32_t rem = idx - t * per_row;
  uint32_t jj = rem / b.cc;
  uint32_t c = rem - jj * b.cc;
  ep = b.ep + (int64_t)t * b.ep_row_stride + (int64_t)jj * b.run_bytes + ((int64_t)c << 4);
  tp_rel = b.tp + (int64_t)t * b.tp_row_stride + ((int64_t)c << 4);
  group = b.g0 + jj;
}

}  // namespace moebius
#endif  // MOEBIUS_UNITS_H_
