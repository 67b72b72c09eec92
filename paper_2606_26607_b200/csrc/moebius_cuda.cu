// moebius_cuda.cu -- the fused reshard kernel for sm_100a and its launch path.
//
// ONE persistent kernel executes the whole work list of a switch (expert-weight slices, KV pages,
// staging copies, scale copies): "reads from the source-mode alias and writes the slice
// into the ... target-mode slot" -- one HBM read and one write per element (Table 1).
// The paper's H200 kernels push slices over NVLink to peers; here the R ranks are regions of one
// allocation, so the same descriptors drive an on-device relayout bounded by HBM bandwidth.
//
// Scheduling: each warp takes unit ids from one global ticket, in list order; a unit is <= one
// shared-memory stage (48 KB by default).  Dependencies (chain links, KV rounds) are device counters.
// Data path (PATH_TMA, the default): the warps move no data; each is a pipe that issues TMA operations
// through two shared-memory stages -- tensor-map boxes (cp.async.bulk.tensor) on the EP side, where the
// box does the run transposition, and contiguous cp.async.bulk copies on the TP side; expert weights,
// KV pages and staged KV pages alike.  Fallback (PATH_LSU: fp8 scale copies, shapes no box fits, or
// moebius_set_tma(ctx, 0, ..)): 16-byte ld.global / st.global with L1 no-allocate, 8 loads in flight per
// lane, lanes on consecutive 16-byte chunks of the EP-side row.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "moebius_host.h"

namespace moebius {

#define MB_UNROLL 8

__device__ __forceinline__ int4 ld16(const char* p) {
  int4 r;
  // plain (coherent) global load, L1 no-allocate: staging bytes are written and re-read inside one
  // launch, so the non-coherent path (ld.global.nc) is not allowed here
  asm volatile("ld.global.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ void st16(char* p, const int4& v) {
  asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};"
               :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ uint32_t ld_acquire(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// EP side is read, every group goes to its `rep` TP ranks.
__device__ __forceinline__ void xbox_ep_to_tp(const Box& b, int64_t rank_stride, uint32_t lane) {
  const uint32_t n = b.nrows * b.J * b.cc;
  for (uint32_t i0 = 0; i0 < n; i0 += 32 * MB_UNROLL) {
    int4 v[MB_UNROLL];
#pragma unroll
    for (int k = 0; k < MB_UNROLL; ++k) {
      uint32_t idx = i0 + k * 32 + lane;
      if (idx < n) {
        char *ep, *tp; uint32_t g;
        box_chunk(b, idx, ep, tp, g);
        v[k] = ld16(ep);
      }
    }
#pragma unroll
    for (int k = 0; k < MB_UNROLL; ++k) {
      uint32_t idx = i0 + k * 32 + lane;
      if (idx < n) {
        char *ep, *tp; uint32_t g;
        box_chunk(b, idx, ep, tp, g);
        tp += (int64_t)(g * b.rep) * rank_stride;
        for (uint32_t r = 0; r < b.rep; ++r) st16(tp + (int64_t)r * rank_stride, v[k]);
      }
    }
  }
}

// TP side is read (one holder per group), EP side written.
__device__ __forceinline__ void xbox_tp_to_ep(const Box& b, int64_t rank_stride, uint32_t lane) {
  const uint32_t n = b.nrows * b.J * b.cc;
  for (uint32_t i0 = 0; i0 < n; i0 += 32 * MB_UNROLL) {
    int4 v[MB_UNROLL];
#pragma unroll
    for (int k = 0; k < MB_UNROLL; ++k) {
      uint32_t idx = i0 + k * 32 + lane;
      if (idx < n) {
        char *ep, *tp; uint32_t g;
        box_chunk(b, idx, ep, tp, g);
        v[k] = ld16(tp + (int64_t)tp_src_rank(g, b.rep, b.owner) * rank_stride);
      }
    }
#pragma unroll
    for (int k = 0; k < MB_UNROLL; ++k) {
      uint32_t idx = i0 + k * 32 + lane;
      if (idx < n) {
        char *ep, *tp; uint32_t g;
        box_chunk(b, idx, ep, tp, g);
        st16(ep, v[k]);
      }
    }
  }
}

__device__ __forceinline__ void lin_copy(const char* src, char* dst, uint64_t bytes, uint32_t lane) {
  const uint32_t n = (uint32_t)(bytes >> 4);
  for (uint32_t i0 = 0; i0 < n; i0 += 32 * MB_UNROLL) {
    int4 v[MB_UNROLL];
#pragma unroll
    for (int k = 0; k < MB_UNROLL; ++k) {
      uint32_t idx = i0 + k * 32 + lane;
      if (idx < n) v[k] = ld16(src + ((uint64_t)idx << 4));
    }
#pragma unroll
    for (int k = 0; k < MB_UNROLL; ++k) {
      uint32_t idx = i0 + k * 32 + lane;
      if (idx < n) st16(dst + ((uint64_t)idx << 4), v[k]);
    }
  }
}

__device__ __forceinline__ void c2d_copy(const C2dDesc& d, char* base, uint32_t lane) {
  const uint32_t per_row = d.run_bytes >> 2;
  const uint32_t n = d.rows * per_row;
  for (uint32_t idx = lane; idx < n; idx += 32) {
    uint32_t r = idx / per_row, c = idx - r * per_row;
    uint32_t v = *(const volatile uint32_t*)(base + d.src_off + (int64_t)r * d.src_stride + 4 * c);
    *(volatile uint32_t*)(base + d.dst_off + (int64_t)r * d.dst_stride + 4 * c) = v;
  }
}

// ---- TMA path (PATH_TMA segments) ---------------------------------------------------------------
// PTX wrappers.  SASS: UTMALDG / UTMASTG (tensor), UBLKCP (bulk), SYNCS (mbarrier).
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, uint32_t n) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(b)), "r"(n));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* b, uint32_t parity) {
  uint32_t ok;
  asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
               : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
  return ok != 0;
}
// A lost transaction would hang the GPU box; trap instead (about 10 s of polling)
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
  for (uint32_t spins = 0; !mbar_try_wait(b, parity); ++spins)
    if (spins > (1u << 28)) __trap();
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t pol = 0) {
  if (pol)
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 :: "r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
  else
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src, uint32_t bytes, uint64_t pol = 0) {
  if (pol)
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
                 :: "l"(dst), "r"(smem_u32(src)), "r"(bytes), "l"(pol) : "memory");
  else
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 :: "l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_5d(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3, int c4, uint64_t* bar, uint64_t pol = 0) {
  if (pol)
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2,%3,%4,%5,%6}], [%7], %8;"
                 :: "r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(smem_u32(bar)), "l"(pol) : "memory");
  else
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2,%3,%4,%5,%6}], [%7];"
                 :: "r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_5d(const CUtensorMap* tm, int c0, int c1, int c2, int c3, int c4, const void* src, uint64_t pol = 0) {
  if (pol)
    asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.tile.bulk_group.L2::cache_hint [%0, {%1,%2,%3,%4,%5}], [%6], %7;"
                 :: "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(smem_u32(src)), "l"(pol) : "memory");
  else
    asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.tile.bulk_group [%0, {%1,%2,%3,%4,%5}], [%6];"
                 :: "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(smem_u32(src)) : "memory");
}
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3, uint64_t* bar, uint64_t pol = 0) {
  if (pol)
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2,%3,%4,%5}], [%6], %7;"
                 :: "r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)), "l"(pol) : "memory");
  else
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2,%3,%4,%5}], [%6];"
                 :: "r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_4d(const CUtensorMap* tm, int c0, int c1, int c2, int c3, const void* src, uint64_t pol = 0) {
  if (pol)
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.tile.bulk_group.L2::cache_hint [%0, {%1,%2,%3,%4}], [%5], %6;"
                 :: "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(src)), "l"(pol) : "memory");
  else
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.tile.bulk_group [%0, {%1,%2,%3,%4}], [%5];"
                 :: "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(src)) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, uint64_t* bar, uint64_t pol = 0) {
  if (pol)
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2,%3,%4}], [%5], %6;"
                 :: "r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)), "l"(pol) : "memory");
  else
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2,%3,%4}], [%5];"
                 :: "r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* tm, int c0, int c1, int c2, const void* src, uint64_t pol = 0) {
  if (pol)
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group.L2::cache_hint [%0, {%1,%2,%3}], [%4], %5;"
                 :: "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(src)), "l"(pol) : "memory");
  else
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group [%0, {%1,%2,%3}], [%4];"
                 :: "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(src)) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" :: "n"(N) : "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait() { asm volatile("cp.async.bulk.wait_group %0;" :: "n"(N) : "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

// One unit through one stage.  Geometry comes from decode_box / the segment, exactly as on the LSU
// path; smem layout of a stage: XT [group][xt_rows][run], LT [row][chunk], KT [pool][group][page][run].
// The whole warp calls these: lane l issues operations l, l+32, ... of the unit (a unit is up to
// pools x groups x replicas bulk copies), so address arithmetic and issue run in parallel.  Bulk
// async-groups are per thread, hence every lane commits and waits on its own groups in lockstep.
struct TmaCtx {
  const DevParams* p;
  const CUtensorMap* tm_w;
  const CUtensorMap* tm_kv;
  const CUtensorMap* tm_stg;
  const CUtensorMap* tm_wtp;
  uint64_t pl, ps;        // L2 cache-hint policies of the loads / the stores (0: none)
};

// Row coordinate (in the staging tensor map) of pool z's copy of staging slot `slot`: the staging
// buffer is an array of EP-page images, slot-major then pool (moebius_units.h, Seg::stg_pools).
__device__ __forceinline__ int stg_row(const Seg& s, const DevParams& p, uint32_t slot, uint32_t z) {
  return (int)((slot * s.stg_pools + (z - s.stg_pool_begin)) * p.page_tokens);
}

// A block-list segment whose EP side is the block's staging slot (in-place path: parked blocks).  Only the
// TP-side box can serve it -- the EP-side tensor map covers the views, not the staging buffer -- so the planner
// puts such a segment on the TMA path only when every unit of it is a whole box.
__device__ __forceinline__ bool staged_ep(const Seg& s) { return s.n_desc != 0 && (s.kv_mode & 1u) != 0; }

__device__ __forceinline__ KvDesc tma_prefetch_desc(const DevParams& p, const Seg& s, uint32_t ul) {
  KvDesc d = {0, 0, 0, 0};
  if (seg_kind(s) == SEG_KV) {
    uint32_t pb, di;
    kv_unit(s, ul, pb, di);
    const int4 v = __ldg((const int4*)(p.kv + s.desc_begin + di));
    d.ep_rank = v.x; d.ep_page = v.y; d.tp_page = v.z; d.ntok_slot = (uint32_t)v.w;
  } else if (seg_kind(s) == SEG_BULK) {                                   // the unit's BulkDesc (two int64 offsets)
    const int4 v = __ldg((const int4*)(p.bulk + s.desc_begin + ul / (s.row_blocks * s.chunks_per_run)));
    d.ep_rank = v.x; d.ep_page = v.y; d.tp_page = v.z; d.ntok_slot = (uint32_t)v.w;
  } else if (seg_kind(s) == SEG_XPOSE && s.n_desc && !s.stg_pools) {    // an irregular block list: the unit's WBlk
    const int4 v = __ldg((const int4*)(p.wblk + s.pool_begin + ul / s.pools_per_unit));
    d.ep_rank = v.x; d.ep_page = v.y; d.tp_page = v.z; d.ntok_slot = (uint32_t)v.w;   // q, row0, nrows, slot
  }
  return d;
}

// The prefetched descriptor of a block-list unit (tma_prefetch_desc stores a WBlk in the KvDesc's 16 bytes).
__device__ __forceinline__ BulkDesc bulk_of(const KvDesc& d) {
  BulkDesc b;
  b.src_off = (int64_t)(((uint64_t)(uint32_t)d.ep_page << 32) | (uint32_t)d.ep_rank);
  b.dst_off = (int64_t)(((uint64_t)d.ntok_slot << 32) | (uint32_t)d.tp_page);
  return b;
}
__device__ __forceinline__ bool has_wblk(const Seg& s) { return s.n_desc != 0 && s.stg_pools == 0; }
__device__ __forceinline__ WBlk wblk_of(const KvDesc& d) {
  return WBlk{(uint32_t)d.ep_rank, (uint32_t)d.ep_page, (uint32_t)d.tp_page, d.ntok_slot};
}

__device__ __forceinline__ void tma_issue_load(const TmaCtx& c, const Seg& s, uint32_t ul, const KvDesc& d, char* stage,
                                               uint64_t* bar, uint32_t lane) {
  const DevParams& p = *c.p;
  if (seg_kind(s) == SEG_BULK) {                      // strided rows -> dense stage [row][piece]
    BulkUnit b;
    decode_bulk(s, p, ul, b, true, bulk_of(d));
    if (lane == 0) mbar_expect_tx(bar, b.nrows * b.piece);
    __syncwarp();
    if (b.src_stride == (int64_t)b.piece) {
      if (lane == 0) bulk_g2s(stage, b.src, b.nrows * b.piece, bar, c.pl);
    } else {
      for (uint32_t t = lane; t < b.nrows; t += 32) bulk_g2s(stage + (size_t)t * b.piece, b.src + (int64_t)t * b.src_stride, b.piece, bar, c.pl);
    }
    return;
  }
  if (seg_kind(s) == SEG_XPOSE) {
    Box b;
    decode_box(s, p, ul, 0, b, has_wblk(s), wblk_of(d));
    if (s.groups_per_unit == s.n_groups) {          // XT
      const uint32_t q = b.q, row0 = b.row0;
      const uint32_t piece = p.xt_rows * s.run_bytes;
      if ((p.xt_mode == 1 || staged_ep(s)) && b.nrows == p.xt_rows) {
        // TP-side box: the stage holds the unit in EP order [row][group][run], so the EP side is ONE
        // contiguous bulk copy and the run transposition happens in the box over the TP views
        // [run/4][rank][row][slot] (full units only: a ragged box would spill into the next rank's rows)
        if (lane == 0) {
          mbar_expect_tx(bar, piece * s.n_groups);
          if (s.ep_is_src) bulk_g2s(stage, b.ep, piece * s.n_groups, bar, c.pl);
          else tma_load_4d(stage, c.tm_wtp, 0, 0, (int)(q * s.rows_total + row0), (int)(s.desc_begin - p.ep_shift), bar, c.pl);
        }
        return;
      }
      if (s.ep_is_src) {
        if (lane == 0) {
          mbar_expect_tx(bar, piece * s.n_groups);   // the box is always delivered whole (rows past the end are zero-filled)
          tma_load_5d(stage, c.tm_w, 0, (int)row0, 0, (int)q, (int)s.desc_begin, bar, c.pl);
        }
      } else {
        const uint32_t bytes = b.nrows * s.run_bytes;
        if (lane == 0) mbar_expect_tx(bar, bytes * s.n_groups);
        __syncwarp();
        for (uint32_t g = lane; g < s.n_groups; g += 32)
          bulk_g2s(stage + (size_t)g * piece, b.tp + (int64_t)g * p.rank_stride, bytes, bar, c.pl);
      }
    } else {                                          // LT: one group, nrows pieces of chunk bytes
      const uint32_t chunk = s.chunk_bytes;
      if (lane == 0) mbar_expect_tx(bar, b.nrows * chunk);
      __syncwarp();
      if (s.ep_is_src) {
        for (uint32_t t = lane; t < b.nrows; t += 32) bulk_g2s(stage + (size_t)t * chunk, b.ep + (int64_t)t * b.ep_row_stride, chunk, bar, c.pl);
      } else if (lane == 0) {
        bulk_g2s(stage, b.tp + (int64_t)b.g0 * p.rank_stride, b.nrows * chunk, bar, c.pl);
      }
    }
    return;
  }
  // KT.  The EP side of a unit is the pool page (KV_MOVE), the staging slot (KV_MOVE_STG), or both
  // (KV_STG_COPY: page -> slot when ep_is_src, slot -> page otherwise); page and slot have the same
  // image, so the same box through either tensor map.
  uint32_t pb, di;
  kv_unit(s, ul, pb, di);
  const uint32_t nb = seg_boxes(s, ul);
  const uint32_t z0 = s.pool_begin + pb * s.pools_per_unit;
  const uint32_t ntok = d.ntok_slot & 0xFFu;
  const uint32_t slot = d.ntok_slot >> 8;
  const bool from_slot = s.kv_mode == KV_MOVE_STG || (s.kv_mode == KV_STG_COPY && !s.ep_is_src);
  if (s.ep_is_src || s.kv_mode == KV_STG_COPY) {
    if (lane == 0) mbar_expect_tx(bar, nb * s.ep_page_bytes);
    __syncwarp();
    for (uint32_t k = lane; k < nb; k += 32) {
      if (from_slot) tma_load_3d(stage + (size_t)k * s.ep_page_bytes, c.tm_stg, 0, stg_row(s, p, slot, z0 + k), 0, bar, c.pl);
      else tma_load_5d(stage + (size_t)k * s.ep_page_bytes, c.tm_kv, 0, (int)(d.ep_page * p.page_tokens), 0, (int)(z0 + k), d.ep_rank, bar, c.pl);
    }
  } else {
    const uint32_t bytes = ntok * s.run_bytes;
    if (lane == 0) mbar_expect_tx(bar, nb * s.n_groups * bytes);
    __syncwarp();
    for (uint32_t o = lane; o < nb * s.n_groups; o += 32) {
      const uint32_t k = o / s.n_groups, g = o - k * s.n_groups;
      const char* src = p.base + s.ep_off + (int64_t)(z0 + k) * s.pool_bytes + (int64_t)d.tp_page * s.tp_page_bytes +
                        (int64_t)tp_src_rank(g, s.rep, d.ep_rank) * p.rank_stride;
      bulk_g2s(stage + (size_t)k * s.ep_page_bytes + (size_t)g * s.tp_page_bytes, src, bytes, bar, c.pl);
    }
  }
}

__device__ __forceinline__ void tma_issue_store(const TmaCtx& c, const Seg& s, uint32_t ul, const KvDesc& d, char* stage,
                                                uint32_t lane) {
  const DevParams& p = *c.p;
  if (seg_kind(s) == SEG_BULK) {
    BulkUnit b;
    decode_bulk(s, p, ul, b, true, bulk_of(d));
    if (b.dst_stride == (int64_t)b.piece) {
      if (lane == 0) bulk_s2g(b.dst, stage, b.nrows * b.piece, c.ps);
    } else {
      for (uint32_t t = lane; t < b.nrows; t += 32) bulk_s2g(b.dst + (int64_t)t * b.dst_stride, stage + (size_t)t * b.piece, b.piece, c.ps);
    }
    bulk_commit();
    return;
  }
  if (seg_kind(s) == SEG_XPOSE) {
    Box b;
    decode_box(s, p, ul, 0, b, has_wblk(s), wblk_of(d));
    if (s.groups_per_unit == s.n_groups) {          // XT
      const uint32_t q = b.q, row0 = b.row0;
      const uint32_t piece = p.xt_rows * s.run_bytes;
      if ((p.xt_mode == 1 || staged_ep(s)) && b.nrows == p.xt_rows) {
        if (lane == 0) {
          if (s.ep_is_src) tma_store_4d(c.tm_wtp, 0, 0, (int)(q * s.rows_total + row0), (int)(s.desc_begin - p.ep_shift), stage, c.ps);
          else bulk_s2g(b.ep, stage, piece * s.n_groups, c.ps);
        }
        bulk_commit();
        return;
      }
      if (s.ep_is_src) {
        const uint32_t bytes = b.nrows * s.run_bytes;
        for (uint32_t g = lane; g < s.n_groups; g += 32)
          bulk_s2g(b.tp + (int64_t)g * p.rank_stride, stage + (size_t)g * piece, bytes, c.ps);
      } else if (lane == 0) {
        tma_store_5d(c.tm_w, 0, (int)row0, 0, (int)q, (int)s.desc_begin, stage, c.ps);   // rows past the end are clipped
      }
    } else {                                          // LT
      const uint32_t chunk = s.chunk_bytes;
      if (s.ep_is_src) {
        if (lane == 0) bulk_s2g(b.tp + (int64_t)b.g0 * p.rank_stride, stage, b.nrows * chunk, c.ps);
      } else {
        for (uint32_t t = lane; t < b.nrows; t += 32) bulk_s2g(b.ep + (int64_t)t * b.ep_row_stride, stage + (size_t)t * chunk, chunk, c.ps);
      }
    }
    bulk_commit();
    return;
  }
  uint32_t pb, di;
  kv_unit(s, ul, pb, di);
  const uint32_t nb = seg_boxes(s, ul);
  const uint32_t z0 = s.pool_begin + pb * s.pools_per_unit;
  const uint32_t ntok = d.ntok_slot & 0xFFu;
  const uint32_t slot = d.ntok_slot >> 8;
  const bool to_slot = (s.kv_mode == KV_MOVE_STG && !s.ep_is_src) || (s.kv_mode == KV_STG_COPY && s.ep_is_src);
  if (s.ep_is_src && s.kv_mode != KV_STG_COPY) {
    const uint32_t bytes = ntok * s.run_bytes;
    const uint32_t per_pool = s.n_groups * s.rep;
    for (uint32_t o = lane; o < nb * per_pool; o += 32) {
      const uint32_t k = o / per_pool, gr = o - k * per_pool, g = gr / s.rep;   // gr = g*rep + r = destination rank
      char* dst = p.base + s.ep_off + (int64_t)(z0 + k) * s.pool_bytes + (int64_t)d.tp_page * s.tp_page_bytes +
                  (int64_t)gr * p.rank_stride;
      bulk_s2g(dst, stage + (size_t)k * s.ep_page_bytes + (size_t)g * s.tp_page_bytes, bytes, c.ps);
    }
  } else {
    // the whole page box is written: slots past the valid tokens get unspecified bytes (reading A10)
    for (uint32_t k = lane; k < nb; k += 32) {
      if (to_slot) tma_store_3d(c.tm_stg, 0, stg_row(s, p, slot, z0 + k), 0, stage + (size_t)k * s.ep_page_bytes, c.ps);
      else tma_store_5d(c.tm_kv, 0, (int)(d.ep_page * p.page_tokens), 0, (int)(z0 + k), d.ep_rank, stage + (size_t)k * s.ep_page_bytes, c.ps);
    }
  }
  bulk_commit();
}

__device__ __forceinline__ void lsu_unit(const Seg& s, const DevParams& p, uint32_t ul, uint32_t lane) {
  if (seg_kind(s) == SEG_COPY2D) {
    c2d_copy(p.c2d[s.desc_begin + ul], p.base, lane);
    return;
  }
  if (seg_kind(s) == SEG_BULK) {
    BulkUnit b;
    decode_bulk(s, p, ul, b);
    for (uint32_t t = 0; t < b.nrows; ++t) lin_copy(b.src + (int64_t)t * b.src_stride, b.dst + (int64_t)t * b.dst_stride, b.piece, lane);
    return;
  }
  const uint32_t nb = seg_boxes(s, ul);
  for (uint32_t k = 0; k < nb; ++k) {
    Box b;
    decode_box(s, p, ul, k, b);
    if (b.lin) lin_copy(b.lin_src, b.lin_dst, b.lin_bytes, lane);
    else if (s.ep_is_src) xbox_ep_to_tp(b, p.rank_stride, lane);
    else xbox_tp_to_ep(b, p.rank_stride, lane);
  }
}

// Every warp is a PIPE: it takes unit tickets in list order and, for PATH_TMA units, runs a software
// pipeline through its private RING in shared memory (ring_bytes per pipe).  A unit takes exactly the
// bytes it needs from the ring, in FIFO order -- 24-KB weight units and 16-KB KV pages pack the same
// 48-KB ring two resp. three deep -- its loads land there (mbarrier), its stores drain from there (bulk
// async-group), and the space returns when the store has read it.  Up to ld_max units of a pipe have
// their loads in flight while the stores of the units before them drain.  Measured on B200: finer units on
// more pipes smooth the read/write mix the DRAM sees (4 pipes x 48-KB ring against 2 pipes x 2 x 48-KB
// stages: weights + 2 %, KV + 1.5-2.5 %), as long as no ring byte stays empty.
// PATH_LSU units are copied by the whole warp.  Before a pipe blocks on a dependency counter it drains its
// own pipeline, so waits can never be circular.
// -DMOEBIUS_PIPE_STATS: every pipe adds up where its time goes (globaltimer ns, lane 0) and the sums land
// in the descriptor buffer's header at bytes 64.. (uint64 each: retire wait, release wait, dependency
// stall, stalls, units, active time, publish wait, ticket wait); the header is zeroed by every moebius_reshard.
#ifdef MOEBIUS_PIPE_STATS
__device__ __forceinline__ uint64_t gtime() { uint64_t t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
#define MB_STAT_T0 const uint64_t stat_t0_ = gtime()
#define MB_STAT_ADD(i) stat_[i] += gtime() - stat_t0_
#define MB_STAT_INC(i) stat_[i] += 1
#else
#define MB_STAT_T0
#define MB_STAT_ADD(i)
#define MB_STAT_INC(i)
#endif
constexpr uint32_t kPipeQ = 8;            // units in flight per pipe (ring entries, mbarriers)
constexpr uint32_t kPipeHdrBytes = 384;   // per pipe: kPipeQ mbarriers + kPipeQ entries
struct PipeEnt {          // 32 bytes: one unit in flight
  uint32_t si, ul, off, size;
  KvDesc   d;
};
static_assert(kPipeQ * 8 + kPipeQ * sizeof(PipeEnt) <= kPipeHdrBytes, "pipe header");

__device__ __forceinline__ void bulk_wait_read_n(uint32_t n) {   // the immediate operand, for n < kPipeQ
  switch (n) {
    case 0: bulk_wait_read<0>(); break;
    case 1: bulk_wait_read<1>(); break;
    case 2: bulk_wait_read<2>(); break;
    case 3: bulk_wait_read<3>(); break;
    case 4: bulk_wait_read<4>(); break;
    case 5: bulk_wait_read<5>(); break;
    case 6: bulk_wait_read<6>(); break;
    default: bulk_wait_read<7>(); break;
  }
}

// Ring bytes a PATH_TMA unit occupies (what its loads deliver), rounded to the 128-byte alignment a
// tensor-map box needs in shared memory.
__device__ __forceinline__ uint32_t tma_unit_bytes(const Seg& s, const DevParams& p, uint32_t ul) {
  uint32_t b;
  if (seg_kind(s) == SEG_KV) b = seg_boxes(s, ul) * s.ep_page_bytes;
  else if (seg_kind(s) == SEG_XPOSE && s.groups_per_unit == s.n_groups) b = p.xt_rows * s.run_bytes * s.n_groups;   // a box is delivered whole
  else b = s.rows_per_unit * s.chunk_bytes;          // LT and BULK: rows x piece
  return (b + 127u) & ~127u;
}

template <int kMinCtasPerSm>   // 1: plans with PATH_TMA segments (shared-memory bound); 2: ld/st-only plans
__global__ void __launch_bounds__(256, kMinCtasPerSm)
moebius_reshard_kernel(const __grid_constant__ DevParams p_in, const __grid_constant__ CUtensorMap tm_w,
                       const __grid_constant__ CUtensorMap tm_kv, const __grid_constant__ CUtensorMap tm_stg,
                       const __grid_constant__ CUtensorMap tm_wtp) {
  extern __shared__ __align__(1024) char smem[];
  // The arguments are the same for every switch of a context (so that the launch can be replayed
  // from a captured graph); what differs per plan is read from the uploaded image's header.
  DevParams p = p_in;
  auto load_hdr = [&](const PlanHdr* hp) {
    const uint4 h = __ldg((const uint4*)hp);
    p.n_segs = h.x;
    p.total_units = h.y;
    p.segs = (const Seg*)((const char*)hp + sizeof(PlanHdr));
    p.kv = (const KvDesc*)((const char*)hp + (int64_t)(int32_t)h.z);     // signed: a wave header sits
    p.c2d = (const C2dDesc*)((const char*)hp + (int64_t)(int32_t)h.w);   // behind the arrays it uses
    p.bulk = (const BulkDesc*)((const char*)hp + (int64_t)(int32_t)__ldg(&hp->bulk_off));
    p.wblk = (const WBlk*)((const char*)hp + (int64_t)(int32_t)__ldg(&hp->wblk_off));
  };
  load_hdr(p_in.hdr);
  // Round-barrier mode: this CTA belongs to one share and walks the plan's dependency waves, each from
  // its own dependency-free segment list and with the share's own ticket; a barrier across ALL shares
  // (this launch's and, on several GPUs, the peers') separates the waves.
  const bool bar_mode = p_in.n_shares > 0;
  uint32_t my_share = 0, share_ctas = 0, n_waves = 1;
  const uint32_t* wave_tab = nullptr;
  if (bar_mode) {
    my_share = p_in.share_first + (uint32_t)(((uint64_t)blockIdx.x * p_in.share_count) / gridDim.x);
    const uint32_t k = my_share - p_in.share_first;     // CTAs [ceil(k*G/n), ceil((k+1)*G/n)) map to share k
    const uint32_t lo = (uint32_t)(((uint64_t)k * gridDim.x + p_in.share_count - 1) / p_in.share_count);
    const uint32_t hi = (uint32_t)(((uint64_t)(k + 1) * gridDim.x + p_in.share_count - 1) / p_in.share_count);
    share_ctas = hi - lo;
    n_waves = __ldg(&p_in.hdr->n_waves);
    wave_tab = (const uint32_t*)((const char*)p_in.hdr + __ldg(&p_in.hdr->wave_tab_off));
    p.rank_lo = p_in.share_bounds[my_share];
    p.rank_hi = p_in.share_bounds[my_share + 1];
  }
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t n_pipes = blockDim.x >> 5;
  uint64_t* bar = (uint64_t*)(smem + (size_t)warp * kPipeHdrBytes);           // kPipeQ barriers per pipe
  PipeEnt* ent = (PipeEnt*)(smem + (size_t)warp * kPipeHdrBytes + kPipeQ * 8);
  const uint32_t hdr_bytes = (n_pipes * kPipeHdrBytes + 1023u) & ~1023u;
  char* ring = smem + hdr_bytes + (size_t)warp * p.ring_bytes;
  if (lane == 0 && p.ring_bytes) {
    for (uint32_t i = 0; i < kPipeQ; ++i) mbar_init(bar + i, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncwarp();
  auto make_policy = [](uint32_t code) -> uint64_t {   // 0 none, 1 evict_first, 2 evict_last, 3 evict_normal, 4 evict_unchanged
    uint64_t pol = 0;
    if (code == 1) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    else if (code == 2) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    else if (code == 3) asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(pol));
    else if (code == 4) asm volatile("createpolicy.fractional.L2::evict_unchanged.b64 %0, 1.0;" : "=l"(pol));
    return pol;
  };
  TmaCtx tc{&p, &tm_w, &tm_kv, &tm_stg, &tm_wtp, make_policy(p.l2_ld), make_policy(p.l2_st)};

#ifdef MOEBIUS_PIPE_STATS
  uint64_t stat_[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  const uint64_t stat_begin_ = gtime();
#endif
  // pipe state; identical in every lane (it depends on uniform values only).  Units in flight are
  // entries [q_tail, q_head) of the FIFO: [q_tail, q_load) have their stores committed (one bulk group
  // each, in this order), [q_load, q_head) their loads in flight.  Entry i uses barrier i % kPipeQ, whose
  // phase parity is (i / kPipeQ) & 1.
  uint32_t q_head = 0, q_load = 0, q_tail = 0;
  uint32_t ring_wr = 0, ring_free = p.ring_bytes;
  const uint32_t ld_max = p.ld_max ? p.ld_max : 2u;
  // Completion signals are batched: units whose store groups are committed but not yet signalled all
  // belong to counter pend_ctr; one fence + one atomicAdd publishes them (a per-unit fence + atomic costs
  // a third of the pipe's time).  When the counter changes the batch is CLOSED but not published at once,
  // which would mean waiting for its last store group: it waits in a short queue (cq_*, oldest first) and
  // is published two units later, when a wait for "all but the two youngest groups" returns at once.
  // Three entries are enough for a counter that changes with every unit (block lists of the in-place
  // path, where a wave of an object is a handful of units per pipe).  A drain publishes everything.
  int32_t pend_ctr = -1;
  uint32_t pend_n = 0;
  int32_t cq_c0 = -1, cq_c1 = -1, cq_c2 = -1;       // scalars, not arrays: they stay in registers
  uint32_t cq_n0 = 0, cq_n1 = 0, cq_n2 = 0, cq_a0 = 0, cq_a1 = 0, cq_len = 0;   // ages of entries 0 and 1 (entry 2 is always the newest)

  auto publish = [&](int32_t ctr, uint32_t n) {   // after every lane's writes of those units have completed
    fence_proxy_async();
    __syncwarp();
    if (lane == 0 && ctr >= 0 && n) { __threadfence(); atomicAdd(p.counters + ctr, n); }
  };
  auto retire = [&]() {                  // oldest loading unit: its loads landed -> issue its stores
    const uint32_t e = q_load % kPipeQ;
    const PipeEnt en = ent[e];
    const Seg& s = p.segs[en.si];
    const int32_t ctr = s.signal_ctr;
    { MB_STAT_T0; if (lane == 0) mbar_wait(bar + e, (q_load / kPipeQ) & 1u); MB_STAT_ADD(0); }
    __syncwarp();
    tma_issue_store(tc, s, en.ul, en.d, ring + en.off, lane);
    ++q_load;
    ++cq_a0; ++cq_a1;
    if (cq_len && cq_a0 >= 2) {          // the oldest closed batch is two groups old: complete, or nearly
      { MB_STAT_T0; bulk_wait<2>(); MB_STAT_ADD(6); }
      while (cq_len && cq_a0 >= 2) {
        publish(cq_c0, cq_n0);
        cq_c0 = cq_c1; cq_n0 = cq_n1; cq_a0 = cq_a1;
        cq_c1 = cq_c2; cq_n1 = cq_n2; cq_a1 = 0;
        --cq_len;
      }
    }
    if (ctr != pend_ctr) {
      if (pend_ctr >= 0 && pend_n) {
        if (cq_len == 3) {               // cannot happen while batches leave at age 2: kept for safety
          bulk_wait<1>();
          publish(cq_c0, cq_n0); publish(cq_c1, cq_n1); publish(cq_c2, cq_n2);
          cq_len = 0;
        }
        if (cq_len == 0) { cq_c0 = pend_ctr; cq_n0 = pend_n; cq_a0 = 0; }
        else if (cq_len == 1) { cq_c1 = pend_ctr; cq_n1 = pend_n; cq_a1 = 0; }
        else { cq_c2 = pend_ctr; cq_n2 = pend_n; }
        ++cq_len;
      }
      pend_ctr = ctr; pend_n = 0;
    }
    ++pend_n;
  };
  auto release = [&]() {                 // oldest storing unit: its stores have read the ring -> space returns
    { MB_STAT_T0; bulk_wait_read_n(q_load - q_tail - 1); MB_STAT_ADD(1); }   // wait_group is per thread: every lane waits for its own stores,
    __syncwarp();                            // and all of them have before any lane refills the space
    ring_free += ent[q_tail % kPipeQ].size;
    ++q_tail;
  };
  auto drain = [&]() {                   // everything this pipe has in flight completes and is signalled
    while (q_load != q_head) retire();
    bulk_wait<0>();
    if (cq_len > 0) publish(cq_c0, cq_n0);
    if (cq_len > 1) publish(cq_c1, cq_n1);
    if (cq_len > 2) publish(cq_c2, cq_n2);
    cq_len = 0;
    publish(pend_ctr, pend_n);
    pend_n = 0;
    q_tail = q_load;
    ring_wr = 0;
    ring_free = p.ring_bytes;
    __syncwarp();
  };
  // The dependency this pipe has already seen satisfied: counter ok_ctr had reached ok_target.  Counters only
  // grow, so every segment that waits for the same counter and no higher a target -- all segments of one
  // wave of an in-place object, all slices of one KV round -- passes without another acquire-load.
  int32_t ok_ctr = -1;
  uint32_t ok_target = 0;
  auto wait_for = [&](const Seg& s, uint32_t si) {   // dependency of a segment (chain links, KV rounds)
    (void)si;
    if (s.wait_ctr < 0 || (s.wait_ctr == ok_ctr && s.wait_target <= ok_target)) return;
    ok_ctr = s.wait_ctr; ok_target = s.wait_target;
    uint32_t ok = 0;
    if (lane == 0) ok = ld_acquire(p.counters + s.wait_ctr) >= s.wait_target;
    ok = __shfl_sync(0xffffffffu, ok, 0);
    if (!ok) {
      MB_STAT_T0;
      MB_STAT_INC(3);
      drain();
      if (lane == 0) {
        for (uint32_t spins = 0; ld_acquire(p.counters + s.wait_ctr) < s.wait_target; ++spins) {
          __nanosleep(200);
          if (spins > (1u << 26)) __trap();
        }
      }
      MB_STAT_ADD(2);
    }
    __syncwarp();
    fence_proxy_async();     // every lane issues TMA reads of what the signalling units wrote
  };
  uint32_t t_next = 0;
  auto fetch = [&]() { if (lane == 0) t_next = atomicAdd(p.ticket, 1u); };

  const bool share = p.rank_hi - p.rank_lo < p.n_ranks;
  for (uint32_t wv = 0; wv < n_waves; ++wv) {
  if (bar_mode) {
    load_hdr((const PlanHdr*)((const char*)p_in.hdr + __ldg(wave_tab + wv)));
    p.ticket = p_in.counters + (size_t)my_share * n_waves + wv;      // wave lists carry no dependency: the counters are free
    ok_ctr = -1;
  }
  uint32_t si = 0;
  fetch();
  // One unit, start to finish on the LSU path, up to its loads on the TMA path.
  auto execute = [&](uint32_t xsi, uint32_t ul) {
    const Seg& s = p.segs[xsi];
    MB_STAT_INC(4);
    if (seg_path(s) == PATH_TMA) {
      const KvDesc d = tma_prefetch_desc(p, s, ul);   // its latency hides behind the wait in retire()
      const uint32_t need = tma_unit_bytes(s, p, ul);
      while (q_head - q_load >= ld_max) retire();     // at most ld_max units of this pipe are loading
      wait_for(s, xsi);
      // space: contiguous in the ring; a unit that does not fit before the end takes the tail as padding
      bool wrap;
      uint32_t pad;
      for (;;) {
        if (q_head == q_tail) { ring_wr = 0; ring_free = p.ring_bytes; }   // nothing in flight: start over
        wrap = ring_wr + need > p.ring_bytes;
        pad = wrap ? p.ring_bytes - ring_wr : 0u;
        if (ring_free >= need + pad && q_head - q_tail < kPipeQ) break;
        if (q_load == q_tail) retire();
        release();
      }
      const uint32_t off = wrap ? 0u : ring_wr;
      ring_wr = off + need;
      ring_free -= need + pad;
      const uint32_t e = q_head % kPipeQ;
      if (lane == 0) {
        PipeEnt en;
        en.si = xsi; en.ul = ul; en.off = off; en.size = need + pad; en.d = d;
        ent[e] = en;
      }
      __syncwarp();
      tma_issue_load(tc, s, ul, d, ring + off, bar + e, lane);
      ++q_head;
      fetch();                 // its latency hides behind the loads just issued
    } else {
      fetch();
      wait_for(s, xsi);
      lsu_unit(s, p, ul, lane);
      if (s.signal_ctr >= 0) {
        __syncwarp();
        if (lane == 0) { __threadfence(); atomicAdd(p.counters + s.signal_ctr, 1u); }
      }
    }
  };
  for (;;) {
    uint32_t u;
    { MB_STAT_T0; u = __shfl_sync(0xffffffffu, t_next, 0); MB_STAT_ADD(7); }
    if (u >= p.total_units) break;
    // units are handed out in increasing order: search forward from the last segment.  The warp looks at the
    // next 32 segments at once (one round trip; plans of many small segments -- block lists of the in-place
    // path, tight-pool rounds -- change segment every few units, and a binary search is a dozen dependent
    // loads each time); only a jump beyond them falls back to the binary search.
    if (si + 1 < p.n_segs) {
      const uint32_t cand = si + 1 + lane;
      const bool le = cand < p.n_segs && __ldg(&p.segs[cand].unit_begin) <= u;
      const uint32_t m = __ballot_sync(0xffffffffu, le);      // unit_begin is non-decreasing: a prefix of ones
      if (m == 0xffffffffu) {
        uint32_t lo = si + 32, hi = p.n_segs - 1;              // last segment whose unit_begin <= u
        while (lo < hi) {
          uint32_t mid = (lo + hi + 1) >> 1;
          if (__ldg(&p.segs[mid].unit_begin) <= u) lo = mid; else hi = mid - 1;
        }
        si = lo;
      } else {
        si += (uint32_t)__popc(m);
      }
    }
    const Seg& s = p.segs[si];
    const uint32_t ul = u - s.unit_begin;
    if (share) {   // rank share: this launch executes only the units of the ranks it owns
      const uint32_t q = unit_ep_rank(s, p, ul);
      if (q < p.rank_lo || q >= p.rank_hi) { fetch(); continue; }
    }
    execute(si, ul);
  }
  drain();
  if (bar_mode) {
    // every pipe of this CTA has drained: its writes of this wave are complete.  The last CTA of the share
    // raises the share's flag; then everybody waits for the flags of all shares.
    __syncthreads();
    if (threadIdx.x == 0) {
      __threadfence_system();
      uint32_t* arrive = p_in.counters + (size_t)(p_in.n_shares + my_share) * n_waves + wv;
      if (atomicAdd(arrive, 1u) + 1 == share_ctas) {
        uint32_t* mine = (uint32_t*)(p_in.base + (int64_t)p_in.share_bounds[my_share] * p_in.rank_stride + p_in.flag_off) + wv;
        asm volatile("st.release.sys.global.u32 [%0], %1;" :: "l"(mine), "r"(1u) : "memory");
      }
      for (uint32_t sh = 0; sh < p_in.n_shares; ++sh) {
        const uint32_t* f = (const uint32_t*)(p_in.base + (int64_t)p_in.share_bounds[sh] * p_in.rank_stride + p_in.flag_off) + wv;
        uint32_t v = 0;
        for (uint32_t spins = 0;; ++spins) {
          asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(f) : "memory");
          if (v) break;
          __nanosleep(100);
          if (spins > (1u << 26)) __trap();     // a share that never arrives must not hang the box
        }
      }
    }
    __syncthreads();
    fence_proxy_async();     // the next wave's TMA reads see what the other shares wrote
  }
  }
#ifdef MOEBIUS_PIPE_STATS
  if (lane == 0) {
    stat_[5] = gtime() - stat_begin_;
    unsigned long long* out = (unsigned long long*)((char*)p_in.ticket + 64);
    for (int i = 0; i < 8; ++i) atomicAdd(out + i, (unsigned long long)stat_[i]);
  }
#endif
}

// Upload images.  A plan's image is read by the async H2D copies of moebius_reshard, so a buffer that
// goes back to the pool keeps the event recorded after its last upload; the next plan that takes the
// buffer waits on that event before overwriting it.
static bool image_fresh(moebius_ctx* x, int64_t cap, ImageBuf* out) {
  out->p = nullptr; out->bytes = cap; out->pinned = false; out->ev = nullptr;
  if (x->has_device) {
    void* p = nullptr;
    if (cudaHostAlloc(&p, (size_t)cap, cudaHostAllocDefault) == cudaSuccess) {
      out->p = (char*)p; out->pinned = true;
      cudaEvent_t e;
      if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess) out->ev = e; else cudaGetLastError();
      return true;
    }
    cudaGetLastError();
  }
  out->p = (char*)malloc((size_t)cap);
  return out->p != nullptr;
}

bool image_acquire(moebius_ctx* x, int64_t bytes, ImageBuf* out) {
  // smallest pooled buffer that fits, preferring one whose last upload has already completed (so that
  // planning the next switch while the current one runs does not wait for the device)
  const size_t none = x->image_pool.size();
  size_t best = none;
  bool best_ready = false;
  for (size_t i = 0; i < x->image_pool.size(); ++i) {
    const ImageBuf& b = x->image_pool[i];
    if (b.bytes < bytes) continue;
    bool ready = !b.ev || cudaEventQuery((cudaEvent_t)b.ev) == cudaSuccess;
    if (!ready) cudaGetLastError();
    if (best == none || (ready && !best_ready) || (ready == best_ready && b.bytes < x->image_pool[best].bytes)) {
      best = i; best_ready = ready;
    }
  }
  if (best != none) {
    *out = x->image_pool[best];
    x->image_pool.erase(x->image_pool.begin() + (long)best);
    if (out->ev && !best_ready && cudaEventSynchronize((cudaEvent_t)out->ev) != cudaSuccess) cudaGetLastError();
    return true;
  }
  if (x->has_device < 0) {
    int ndev = 0;
    x->has_device = (cudaGetDeviceCount(&ndev) == cudaSuccess && ndev > 0) ? 1 : 0;
    cudaGetLastError();
  }
  // round up so that plans of slightly different sizes share buffers
  const int64_t cap = (bytes + (1 << 20) - 1) >> 20 << 20;
  if (!image_fresh(x, cap, out)) return false;
  // pinning memory can wait for the device: allocate a twin now, so that two plans can be alive
  // (one executing, one being built) without another allocation later
  if (out->pinned && x->image_pool.empty()) {
    ImageBuf twin;
    if (image_fresh(x, cap, &twin)) x->image_pool.push_back(twin);
  }
  return true;
}

void image_free(const ImageBuf& b) {
  if (!b.p) return;
  if (b.ev) { cudaEventSynchronize((cudaEvent_t)b.ev); cudaEventDestroy((cudaEvent_t)b.ev); }
  if (b.pinned) cudaFreeHost(b.p); else free(b.p);
}

void image_release(moebius_ctx* x, const ImageBuf& b) {
  if (!b.p) return;
  if (x->image_pool.size() < 4) x->image_pool.push_back(b); else image_free(b);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// The two tensor maps of the TMA path, over the caller's bound allocation (uint32 elements):
//   weights (gate/up slots):  [run/4][rows = E/R*H][group R][rank R][slot 3L+1], box [run/4][xt_rows][R][1][1]
//   KV (EP pools):            [run/4][rows = pages_ep*pg][group G][pool 2L][rank R], box [run/4][pg][G][1][1]
// Dimension 1 (rows) has the LARGER stride and dimension 2 (group) the smaller one, so a box lands
// in shared memory as [group][row][run]: the run transposition is done by the TMA engine.
static int encode_tmaps(moebius_ctx* x) {
  static_assert(sizeof(CUtensorMap) <= sizeof(x->tmap_w), "CUtensorMap storage");
  memset(x->tmap_w, 0, sizeof(x->tmap_w));
  memset(x->tmap_kv, 0, sizeof(x->tmap_kv));
  memset(x->tmap_stg, 0, sizeof(x->tmap_stg));
  memset(x->tmap_wtp, 0, sizeof(x->tmap_wtp));
  x->tmaps_valid = true;
  if (!x->use_tma || (!x->xt_ok && !x->kt_ok)) return MOEBIUS_OK;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) {
    cudaGetLastError();
    x->tmaps_valid = false;
    return MOEBIUS_E_CUDA;
  }
  EncodeTiledFn enc = (EncodeTiledFn)fn;
  const moebius_config_t& c = x->cfg;
  const cuuint32_t ones[5] = {1, 1, 1, 1, 1};
  if (x->xt_ok) {
    const cuuint64_t run = (cuuint64_t)(c.I / c.R) * x->wb;
    cuuint64_t dims[5] = {run / 4, (cuuint64_t)(c.E / c.R) * c.H, (cuuint64_t)c.R, (cuuint64_t)c.R,
                          (cuuint64_t)(3 * c.L + x->ep_shift)};
    cuuint64_t strides[4] = {run * c.R, run, (cuuint64_t)x->rank_stride, (cuuint64_t)x->S};
    cuuint32_t box[5] = {(cuuint32_t)(run / 4), (cuuint32_t)x->xt_rows, (cuuint32_t)c.R, 1, 1};
    if (enc((CUtensorMap*)x->tmap_w, CU_TENSOR_MAP_DATA_TYPE_UINT32, 5, x->base + x->w_off, dims, strides, box, ones,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) { x->tmaps_valid = false; return MOEBIUS_E_CUDA; }
  }
  if (x->xt_ok) {   // the TP views of the same slots: [run/4][rank R][row R*rows][slot], box [run/4][R][xt_rows][1]
    const cuuint64_t run = (cuuint64_t)(c.I / c.R) * x->wb;
    cuuint64_t dims[4] = {run / 4, (cuuint64_t)c.R, (cuuint64_t)c.E * c.H, (cuuint64_t)(3 * c.L + x->ep_shift)};
    cuuint64_t strides[3] = {(cuuint64_t)x->rank_stride, run, (cuuint64_t)x->S};
    cuuint32_t box[4] = {(cuuint32_t)(run / 4), (cuuint32_t)c.R, (cuuint32_t)x->xt_rows, 1};
    const CUtensorMapL2promotion promo = x->xt_promo == 1 ? CU_TENSOR_MAP_L2_PROMOTION_L2_64B : x->xt_promo == 2 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B
                                        : x->xt_promo == 3 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B : CU_TENSOR_MAP_L2_PROMOTION_NONE;
    if (enc((CUtensorMap*)x->tmap_wtp, CU_TENSOR_MAP_DATA_TYPE_UINT32, 4, x->base + x->w_off, dims, strides, box, ones,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, promo,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) { x->tmaps_valid = false; return MOEBIUS_E_CUDA; }
  }
  if (x->kt_ok) {
    const cuuint64_t run = (cuuint64_t)x->run_kv;
    cuuint64_t dims[5] = {run / 4, (cuuint64_t)x->pages_ep * c.page_tokens, (cuuint64_t)x->G, (cuuint64_t)(2 * c.L),
                          (cuuint64_t)c.R};
    cuuint64_t strides[4] = {run * x->G, run, (cuuint64_t)x->pool_bytes, (cuuint64_t)x->rank_stride};
    cuuint32_t box[5] = {(cuuint32_t)(run / 4), (cuuint32_t)c.page_tokens, (cuuint32_t)x->G, 1, 1};
    if (x->pages_ep < 1 ||
        enc((CUtensorMap*)x->tmap_kv, CU_TENSOR_MAP_DATA_TYPE_UINT32, 5, x->base + x->kv_off, dims, strides, box, ones,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) { x->tmaps_valid = false; return MOEBIUS_E_CUDA; }
  }
  // staging buffer = an array of EP-page images: [run/4][rows = slots*pg][group G], the same box
  if (x->kt_ok && x->staging_bytes >= x->ep_page_bytes && x->stg) {
    const cuuint64_t run = (cuuint64_t)x->run_kv;
    cuuint64_t dims[3] = {run / 4, (cuuint64_t)(x->staging_bytes / x->ep_page_bytes) * c.page_tokens, (cuuint64_t)x->G};
    cuuint64_t strides[2] = {run * x->G, run};
    cuuint32_t box[3] = {(cuuint32_t)(run / 4), (cuuint32_t)c.page_tokens, (cuuint32_t)x->G};
    if (dims[1] > (1ull << 31) ||
        enc((CUtensorMap*)x->tmap_stg, CU_TENSOR_MAP_DATA_TYPE_UINT32, 3, x->stg, dims, strides, box, ones,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) { x->tmaps_valid = false; return MOEBIUS_E_CUDA; }
  }
  return MOEBIUS_OK;
}

void cuda_ctx_destroy(moebius_ctx* x) {
  for (const ImageBuf& b : x->image_pool) image_free(b);
  x->image_pool.clear();
  if (x->mailbox) { cudaFreeHost(x->mailbox); x->mailbox = nullptr; }
  if (x->ev_valid) {
    for (int i = 0; i < 2 * kTimingRing; ++i) cudaEventDestroy((cudaEvent_t)x->ev[i]);
    x->ev_valid = false;
  }
}

}  // namespace moebius

using namespace moebius;

namespace moebius {

// One-off device-side setup of a bound context: device facts, the timing-event ring, the driver entry
// point + the three tensor maps, and the kernel's dynamic shared-memory attribute.  Called by
// moebius_bind and again by moebius_set_tma (the stage geometry changes the maps and the attribute), so
// that moebius_reshard / _staged / _share find everything in place: they create no event, resolve no
// symbol, encode no descriptor and set no attribute.
static size_t pipe_smem_bytes(const moebius_ctx* x) {   // per-pipe headers (barriers + FIFO entries), then the rings
  return (((size_t)x->n_pipes * kPipeHdrBytes + 1023) & ~(size_t)1023) + (size_t)x->n_pipes * (size_t)x->ring_bytes;
}

int device_prepare(moebius_ctx* x) {
  x->prepared = false;
  if (!x->bound) return MOEBIUS_OK;
  if (x->has_device < 0) {
    int ndev = 0;
    x->has_device = (cudaGetDeviceCount(&ndev) == cudaSuccess && ndev > 0) ? 1 : 0;
    cudaGetLastError();
  }
  if (!x->has_device) return MOEBIUS_OK;
  if (x->n_sm == 0) {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return MOEBIUS_E_CUDA;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return MOEBIUS_E_CUDA;
    x->n_sm = n;
  }
  if (!x->ev_valid) {
    for (int i = 0; i < 2 * kTimingRing; ++i) {
      cudaEvent_t e;
      if (cudaEventCreate(&e) != cudaSuccess) {
        for (int k = 0; k < i; ++k) cudaEventDestroy((cudaEvent_t)x->ev[k]);
        return MOEBIUS_E_CUDA;
      }
      x->ev[i] = e;
    }
    x->ev_valid = true;
  }
  if (int rc = encode_tmaps(x)) return rc;
  const bool tma = x->use_tma != 0;   // bulk copies (long runs, attention shards, parked blocks) need the pipes' rings too
  if (tma) {
    const size_t smem = pipe_smem_bytes(x);
    if (cudaFuncSetAttribute(moebius_reshard_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
      cudaGetLastError();
      return MOEBIUS_E_CUDA;
    }
    x->smem_set = smem;
  }
  {  // lazy module loading would otherwise hit the first switch: resolve both kernel variants now
    cudaFuncAttributes fa;
    if (cudaFuncGetAttributes(&fa, moebius_reshard_kernel<1>) != cudaSuccess ||
        cudaFuncGetAttributes(&fa, moebius_reshard_kernel<2>) != cudaSuccess) { cudaGetLastError(); return MOEBIUS_E_CUDA; }
  }
  x->prepared = true;
  return MOEBIUS_OK;
}

}  // namespace moebius

extern "C" int moebius_bind(moebius_ctx_t* x, void* dev_base, void* dev_staging, void* dev_desc,
                            int32_t* dev_tables, moebius_mode_t initial_mode) {
  if (!x || !dev_base || !dev_desc || !dev_tables) return MOEBIUS_E_INVAL;
  if (x->staging_bytes > 0 && !dev_staging) return MOEBIUS_E_INVAL;
  if (initial_mode != MOEBIUS_TP && initial_mode != MOEBIUS_EP) return MOEBIUS_E_INVAL;
  if (((uintptr_t)dev_base | (uintptr_t)dev_staging | (uintptr_t)dev_desc | (uintptr_t)dev_tables) & 255)
    return MOEBIUS_E_INVAL;
  x->base = (char*)dev_base;
  x->stg = (char*)dev_staging;
  x->desc = (char*)dev_desc;
  x->tables = dev_tables;
  x->active_mode = initial_mode;
  x->bound = true;
  x->tmaps_valid = false;
  x->prepared = false;
  // Everything a first switch would otherwise have to set up is done here (the switch
  // path itself allocates nothing).  Without a CUDA device the context stays usable for the host-only
  // planner calls; moebius_reshard then returns MOEBIUS_E_CUDA.
  return device_prepare(x);
}

extern "C" int moebius_set_timing(moebius_ctx_t* x, int enable) {
  if (!x) return MOEBIUS_E_INVAL;
  x->timing = enable ? 1 : 0;
  return MOEBIUS_OK;
}

extern "C" int moebius_kernel_ms_history(moebius_ctx_t* x, float* out_ms, int cap, int* n_out) {
  if (!x || !out_ms || !n_out || cap < 0) return MOEBIUS_E_INVAL;
  *n_out = 0;
  if (!x->ev_valid || x->ev_count == 0) return MOEBIUS_E_STATE;
  int64_t n = x->ev_count < kTimingRing ? x->ev_count : kTimingRing;
  if (n > cap) n = cap;
  for (int64_t i = 0; i < n; ++i) {
    int64_t k = (x->ev_count - n + i) % kTimingRing;
    cudaEvent_t a = (cudaEvent_t)x->ev[2 * k], b = (cudaEvent_t)x->ev[2 * k + 1];
    if (cudaEventSynchronize(b) != cudaSuccess) return MOEBIUS_E_CUDA;
    if (cudaEventElapsedTime(out_ms + i, a, b) != cudaSuccess) return MOEBIUS_E_CUDA;
  }
  *n_out = (int)n;
  return MOEBIUS_OK;
}

extern "C" int moebius_last_kernel_ms(moebius_ctx_t* x, float* ms) {
  if (!x || !ms) return MOEBIUS_E_INVAL;
  int n = 0;
  return moebius_kernel_ms_history(x, ms, 1, &n);
}

namespace {

// What must hold before anything is enqueued: a CUDA device, the one-off setup of device_prepare, and a
// plan built for the current stage geometry (moebius_set_tma after moebius_plan invalidates the plan).
int ready_to_launch(const moebius_ctx* x, const moebius_plan_t* P) {
  if (!x->has_device || !x->prepared) return x->has_device ? MOEBIUS_E_STATE : MOEBIUS_E_CUDA;
  if (P && P->uses_tma && (P->stage_bytes != x->stage_bytes || P->xt_rows != x->xt_rows)) return MOEBIUS_E_STATE;
  if (P && (kSegOff + P->image_bytes > x->desc_bytes || P->tbl_bytes > x->table_bytes)) return MOEBIUS_E_INVAL;
  return MOEBIUS_OK;
}

// Launches the reshard kernel over the image that sits at dev_desc + kSegOff.  `tma`: the variant with
// the pipes' shared-memory rings (it also executes PATH_LSU segments).  `unit_hint` > 0 caps the grid
// for small plans; 0 = the full persistent grid (plan-independent: what a captured graph needs).
struct ShareLaunch {       // round-barrier mode of the kernel (DevParams::n_shares)
  int n_shares, first, count;
  const int32_t* bounds;   // [n_shares + 1]
};

int launch_reshard_kernel(moebius_ctx* x, bool tma, int64_t unit_hint, cudaStream_t st, int64_t hdr_off = 0,
                          int rank_lo = 0, int rank_hi = -1, const ShareLaunch* sl = nullptr) {
  DevParams p;
  memset(&p, 0, sizeof(p));
  if (sl) {
    p.n_shares = (uint32_t)sl->n_shares; p.share_first = (uint32_t)sl->first; p.share_count = (uint32_t)sl->count;
    p.flag_off = x->flag_off;
    for (int i = 0; i <= sl->n_shares; ++i) p.share_bounds[i] = (uint8_t)sl->bounds[i];
  }
  p.base = x->base;
  p.stg = x->stg;
  p.hdr = (const PlanHdr*)(x->desc + kSegOff + hdr_off);
  p.n_ranks = (uint32_t)x->cfg.R;
  p.rank_lo = (uint32_t)rank_lo;
  p.rank_hi = (uint32_t)(rank_hi < 0 ? x->cfg.R : rank_hi);
  p.ticket = (uint32_t*)x->desc;
  p.counters = (uint32_t*)(x->desc + kCtrOff);
  p.rank_stride = x->rank_stride;
  p.wstg_off = x->staging_bytes - x->w_stg_bytes;
  p.xt_mode = (uint32_t)x->xt_mode;
  p.ep_shift = (uint32_t)x->ep_shift;
  p.page_tokens = (uint32_t)x->cfg.page_tokens;
  int threads, per_sm;
  size_t smem = 0;
  if (tma) {
    // one CTA per SM, n_pipes warps, each with two private stages (tensor maps and the shared-memory
    // attribute were set up by device_prepare)
    p.stage_bytes = (uint32_t)x->stage_bytes;
    p.ring_bytes = (uint32_t)x->ring_bytes;
    p.ld_max = (uint32_t)x->ld_max;
    p.l2_ld = (uint32_t)x->l2_ld; p.l2_st = (uint32_t)x->l2_st;
    p.xt_rows = (uint32_t)x->xt_rows;
    threads = 32 * x->n_pipes;
    per_sm = 1;
    smem = pipe_smem_bytes(x);
    if (smem != x->smem_set || !x->tmaps_valid) return MOEBIUS_E_STATE;
  } else {
    threads = x->threads > 0 ? x->threads : 256;
    per_sm = x->ctas_per_sm > 0 ? x->ctas_per_sm : 2;
  }
  int64_t grid = (int64_t)x->n_sm * per_sm;
  if (unit_hint > 0) {
    int64_t grid_cap = (unit_hint + threads / 32 - 1) / (threads / 32);
    if (grid > grid_cap) grid = grid_cap;
  }
  if (sl) {
    // CTAs of different shares wait for one another: all of them must be resident at once, which only
    // a cooperative launch guarantees (one CTA per SM with the pipes' rings, two without)
    void* args[5] = {(void*)&p, (void*)x->tmap_w, (void*)x->tmap_kv, (void*)x->tmap_stg, (void*)x->tmap_wtp};
    const void* fn = tma ? (const void*)moebius_reshard_kernel<1> : (const void*)moebius_reshard_kernel<2>;
    if (grid < sl->count) return MOEBIUS_E_INVAL;
    return cudaLaunchCooperativeKernel(fn, dim3((unsigned)grid), dim3((unsigned)threads), args, smem, st) == cudaSuccess
               ? MOEBIUS_OK : MOEBIUS_E_CUDA;
  }
  if (tma)
    moebius_reshard_kernel<1><<<(unsigned)grid, threads, smem, st>>>(p, *(const CUtensorMap*)x->tmap_w, *(const CUtensorMap*)x->tmap_kv,
                                                                     *(const CUtensorMap*)x->tmap_stg, *(const CUtensorMap*)x->tmap_wtp);
  else
    moebius_reshard_kernel<2><<<(unsigned)grid, threads, 0, st>>>(p, *(const CUtensorMap*)x->tmap_w, *(const CUtensorMap*)x->tmap_kv,
                                                                  *(const CUtensorMap*)x->tmap_stg, *(const CUtensorMap*)x->tmap_wtp);
  return cudaGetLastError() == cudaSuccess ? MOEBIUS_OK : MOEBIUS_E_CUDA;
}

}  // namespace

extern "C" int moebius_reshard(moebius_ctx_t* x, const moebius_plan_t* P, void* cuda_stream) {
  if (!x || !P || P->ctx != x) return MOEBIUS_E_INVAL;
  if (!x->bound || x->active_mode != P->from) return MOEBIUS_E_STATE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // Every check comes before the first enqueue: a call that fails here has touched nothing.  (A CUDA
  // error returned by one of the enqueues below is a sticky device fault, not a recoverable state.)
  if (int rc = ready_to_launch(x, P)) return rc;
  cudaEvent_t ev_a = nullptr, ev_b = nullptr;
  if (x->timing) {
    int64_t k = x->ev_count % kTimingRing;
    ev_a = (cudaEvent_t)x->ev[2 * k]; ev_b = (cudaEvent_t)x->ev[2 * k + 1];
  }
  // 1. work list -> device; ticket and the counters this plan uses -> 0
  if (cudaMemsetAsync(x->desc, 0, (size_t)(kCtrOff + 4 * (int64_t)(P->n_counters ? P->n_counters : 1)), st) != cudaSuccess)
    return MOEBIUS_E_CUDA;
  if (cudaMemcpyAsync(x->desc + kSegOff, P->image, (size_t)P->image_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess)
    return MOEBIUS_E_CUDA;
  // 2. the kernel
  if (x->timing) cudaEventRecord(ev_a, st);
  if (P->total_units) {
    if (int rc = launch_reshard_kernel(x, P->uses_tma, (int64_t)P->total_units, st)) return rc;
  }
  if (x->timing) { cudaEventRecord(ev_b, st); x->ev_count++; }
  // 3. publish: new tables, owner vector and the active-mode flag at their fixed address
  if (cudaMemcpyAsync(x->tables, P->tbl_image, (size_t)P->tbl_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess)
    return MOEBIUS_E_CUDA;
  if (P->buf.ev && cudaEventRecord((cudaEvent_t)P->buf.ev, st) != cudaSuccess) return MOEBIUS_E_CUDA;
  x->active_mode = P->to;
  x->switch_count++;
  return MOEBIUS_OK;
}

// ---- the switch as a graph-capturable, plan-independent sequence ------------------------------------
extern "C" int moebius_stage_plan(moebius_ctx_t* x, const moebius_plan_t* P) {
  if (!x || !P || P->ctx != x) return MOEBIUS_E_INVAL;
  if (!x->bound || x->active_mode != P->from) return MOEBIUS_E_STATE;
  if (int rc = ready_to_launch(x, P)) return rc;
  const int64_t img_cap = x->desc_bytes - kSegOff;
  if (P->image_bytes > img_cap || P->tbl_bytes > x->table_bytes) return MOEBIUS_E_INVAL;
  if (!x->mailbox) {
    void* m = nullptr;
    if (cudaHostAlloc(&m, (size_t)(img_cap + x->table_bytes), cudaHostAllocDefault) != cudaSuccess) {
      cudaGetLastError();
      return MOEBIUS_E_CUDA;
    }
    memset(m, 0, (size_t)(img_cap + x->table_bytes));
    x->mailbox = (char*)m;
  }
  memcpy(x->mailbox, P->image, (size_t)P->image_bytes);
  memcpy(x->mailbox + img_cap, P->tbl_image, (size_t)P->tbl_bytes);
  x->active_mode = P->to;
  x->switch_count++;
  return MOEBIUS_OK;
}

extern "C" int moebius_reshard_staged(moebius_ctx_t* x, void* cuda_stream) {
  if (!x) return MOEBIUS_E_INVAL;
  if (!x->bound || !x->mailbox) return MOEBIUS_E_STATE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (int rc = ready_to_launch(x, nullptr)) return rc;
  const int64_t img_cap = x->desc_bytes - kSegOff;
  // every size, address and launch dimension below is the same for every plan of this context
  if (cudaMemsetAsync(x->desc, 0, (size_t)kSegOff, st) != cudaSuccess) return MOEBIUS_E_CUDA;
  if (cudaMemcpyAsync(x->desc + kSegOff, x->mailbox, (size_t)img_cap, cudaMemcpyHostToDevice, st) != cudaSuccess)
    return MOEBIUS_E_CUDA;
  const bool tma = x->use_tma != 0;   // bulk copies (long runs, attention shards, parked blocks) need the pipes' rings too
  if (int rc = launch_reshard_kernel(x, tma, 0, st)) return rc;
  if (cudaMemcpyAsync(x->tables, x->mailbox + img_cap, (size_t)x->table_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess)
    return MOEBIUS_E_CUDA;
  return MOEBIUS_OK;
}

// ---- rank-share execution: the plan wave by wave, each launch restricted to a range of ranks -------
extern "C" int moebius_plan_waves(const moebius_plan_t* P, int32_t* n_waves) {
  if (!P || !n_waves) return MOEBIUS_E_INVAL;
  *n_waves = P->n_waves;
  return MOEBIUS_OK;
}

extern "C" int moebius_reshard_share(moebius_ctx_t* x, const moebius_plan_t* P, int rank_lo, int rank_hi, int wave,
                                     void* cuda_stream) {
  if (!x || !P || P->ctx != x) return MOEBIUS_E_INVAL;
  if (rank_lo < 0 || rank_hi > x->cfg.R || rank_lo >= rank_hi || wave < 0 || wave >= P->n_waves) return MOEBIUS_E_INVAL;
  if (!x->bound || x->active_mode != P->from) return MOEBIUS_E_STATE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (int rc = ready_to_launch(x, P)) return rc;
  if (wave == 0) {   // the work list (all waves) goes up once, with the first wave
    if (cudaMemcpyAsync(x->desc + kSegOff, P->image, (size_t)P->image_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess)
      return MOEBIUS_E_CUDA;
    if (P->buf.ev && cudaEventRecord((cudaEvent_t)P->buf.ev, st) != cudaSuccess) return MOEBIUS_E_CUDA;
  }
  if (cudaMemsetAsync(x->desc, 0, (size_t)kHdrBytes, st) != cudaSuccess) return MOEBIUS_E_CUDA;   // the ticket
  if (P->wave_units[(size_t)wave] == 0) return MOEBIUS_OK;
  return launch_reshard_kernel(x, P->uses_tma, (int64_t)P->wave_units[(size_t)wave], st, P->wave_hdr_off[(size_t)wave],
                               rank_lo, rank_hi);
}

extern "C" int moebius_reshard_publish(moebius_ctx_t* x, const moebius_plan_t* P, void* cuda_stream) {
  if (!x || !P || P->ctx != x) return MOEBIUS_E_INVAL;
  if (!x->bound || x->active_mode != P->from) return MOEBIUS_E_STATE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (int rc = ready_to_launch(x, P)) return rc;
  if (cudaMemcpyAsync(x->tables, P->tbl_image, (size_t)P->tbl_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess)
    return MOEBIUS_E_CUDA;
  if (P->buf.ev && cudaEventRecord((cudaEvent_t)P->buf.ev, st) != cudaSuccess) return MOEBIUS_E_CUDA;
  x->active_mode = P->to;
  x->switch_count++;
  return MOEBIUS_OK;
}

// ---- the switch as ONE launch per GPU with a device-side round barrier --------------------------------
extern "C" int moebius_reshard_shares(moebius_ctx_t* x, const moebius_plan_t* P, int n_shares, const int32_t* rank_bounds,
                                      int share_first, int share_count, void* cuda_stream) {
  if (!x || !P || P->ctx != x || !rank_bounds) return MOEBIUS_E_INVAL;
  const int R = x->cfg.R;
  if (n_shares < 1 || n_shares > R || share_first < 0 || share_count < 1 || share_first + share_count > n_shares) return MOEBIUS_E_INVAL;
  if (rank_bounds[0] != 0 || rank_bounds[n_shares] != R) return MOEBIUS_E_INVAL;
  for (int i = 0; i < n_shares; ++i) if (rank_bounds[i + 1] <= rank_bounds[i]) return MOEBIUS_E_INVAL;
  if (!x->bound || x->active_mode != P->from) return MOEBIUS_E_STATE;
  if (int rc = ready_to_launch(x, P)) return rc;
  if (2 * (int64_t)n_shares * P->n_waves > kMaxCounters || P->n_waves > kMaxCounters) return MOEBIUS_E_INVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // tickets (one per share and wave) and arrival counters live in the counter area; the flag pages of
  // the shares THIS launch executes are cleared here -- on several GPUs every process clears its own and
  // a host barrier precedes the launches (one per switch, not one per wave)
  if (cudaMemsetAsync(x->desc, 0, (size_t)kSegOff, st) != cudaSuccess) return MOEBIUS_E_CUDA;
  for (int sh = share_first; sh < share_first + share_count; ++sh)
    if (P->n_waves && cudaMemsetAsync(x->base + (int64_t)rank_bounds[sh] * x->rank_stride + x->flag_off, 0, (size_t)P->n_waves * 4, st) != cudaSuccess)
      return MOEBIUS_E_CUDA;
  if (cudaMemcpyAsync(x->desc + kSegOff, P->image, (size_t)P->image_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess)
    return MOEBIUS_E_CUDA;
  if (P->buf.ev && cudaEventRecord((cudaEvent_t)P->buf.ev, st) != cudaSuccess) return MOEBIUS_E_CUDA;
  cudaEvent_t ev_a = nullptr, ev_b = nullptr;
  if (x->timing) {
    int64_t k = x->ev_count % kTimingRing;
    ev_a = (cudaEvent_t)x->ev[2 * k]; ev_b = (cudaEvent_t)x->ev[2 * k + 1];
    cudaEventRecord(ev_a, st);
  }
  if (P->total_units) {
    ShareLaunch sl{n_shares, share_first, share_count, rank_bounds};
    if (int rc = launch_reshard_kernel(x, P->uses_tma, 0, st, 0, 0, -1, &sl)) return rc;
  }
  if (x->timing) { cudaEventRecord(ev_b, st); x->ev_count++; }
  return MOEBIUS_OK;   // the caller ends the switch with moebius_reshard_publish, as on the wave-by-wave path
}
