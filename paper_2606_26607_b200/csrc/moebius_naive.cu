// moebius_naive.cu -- the STAGED comparison path of PAPER.md:162-170 and Table 1 (:176-189), on one device.
//
// The paper's "Naive" implementation maps a switch onto collectives: per layer, gather the source bytes
// into per-peer chunks in a staging buffer (local permute), exchange the chunks (All-to-All), and --
// for the paged KV cache -- scatter the received chunks into the target pages.  Table 1 counts its HBM
// passes per element: weights 2 reads + 1 write (+ the receiver's write, folded into the NVLink
// column), cache 3 + 2, against 1 + 0 for the direct kernel.  Here the R ranks are regions of one
// device, so the exchange is a device copy and the receiver's write is an HBM write as well:
//   weights   permute (1R + 1W) + exchange (1R + 1W)                      = 2 x the direct path's traffic
//   KV cache  gather (1R + 1W) + exchange (1R + 1W) + scatter (1R + 1W)   = 3 x
// The result is bit-identical to moebius_reshard (same plan, same target views, same tables); it exists
// so that the pass counts of Table 1 can be MEASURED next to the fused kernel (ncu dram__bytes per
// switch) and the fused kernel's gain timed on the same box.  Plain ld.global/st.global kernels, one
// launch per stage and object/pool, like the per-layer staging the paper describes.  Not on the
// product path: nothing else in the library calls into this file.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <vector>

#include "moebius_host.h"

namespace moebius {

namespace {

__device__ __forceinline__ int4 nld16(const char* p) {
  int4 r;
  asm volatile("ld.global.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ void nst16(char* p, const int4& v) {
  asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};" :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// n0 x n1 x n2 runs of `run16` 16-byte chunks, each side with its own three strides (bytes)
struct Copy4 {
  const char* src;
  char* dst;
  int64_t ss[3], ds[3];
  uint32_t n[3];
  uint32_t run16;
};

// blockIdx.y = (i0, i1); blockIdx.x strides over the n2 x run16 chunks of that pair (32-bit index math)
__global__ void __launch_bounds__(256) naive_copy4d_kernel(const Copy4 c) {
  const uint32_t a0 = blockIdx.y / c.n[1], i1 = blockIdx.y - a0 * c.n[1];
  const char* src0 = c.src + a0 * c.ss[0] + i1 * c.ss[1];
  char* dst0 = c.dst + a0 * c.ds[0] + i1 * c.ds[1];
  const uint32_t inner = c.n[2] * c.run16;
  const uint32_t step = gridDim.x * blockDim.x;
  for (uint32_t i0 = blockIdx.x * blockDim.x + threadIdx.x; i0 < inner; i0 += 4 * step) {
    int4 v[4];
    char* d[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t i = i0 + k * step;
      if (i < inner && i >= i0) {
        const uint32_t i2 = i / c.run16, ch = i - i2 * c.run16;
        d[k] = dst0 + i2 * c.ds[2] + ((int64_t)ch << 4);
        v[k] = nld16(src0 + i2 * c.ss[2] + ((int64_t)ch << 4));
      }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t i = i0 + k * step;
      if (i < inner && i >= i0) nst16(d[k], v[k]);
    }
  }
}

// rows x run16 chunks per descriptor; side A is the pool (or any strided place), side B the buffer
struct RowsDesc {
  int64_t a_off, b_off;        // bytes from the two bases the launch names
  uint32_t rows, run16, a_stride, b_stride;
};
static_assert(sizeof(RowsDesc) == 32, "RowsDesc must be 32 bytes");

// one block per descriptor slice: blockIdx.x = descriptor, blockIdx.y strides over its chunks
__global__ void __launch_bounds__(128) naive_rows_kernel(const RowsDesc* descs, char* a_base, char* b_base, int a_to_b) {
  const RowsDesc d = descs[blockIdx.x];
  const uint32_t total = d.rows * d.run16;
  for (uint32_t i = blockIdx.y * blockDim.x + threadIdx.x; i < total; i += gridDim.y * blockDim.x) {
    const uint32_t r = i / d.run16, ch = i - r * d.run16;
    char* a = a_base + d.a_off + (int64_t)r * d.a_stride + ((int64_t)ch << 4);
    char* b = b_base + d.b_off + (int64_t)r * d.b_stride + ((int64_t)ch << 4);
    if (a_to_b) nst16(b, nld16(a)); else nst16(a, nld16(b));
  }
}

// 4-byte granular 2-D copies (fp8 block scales): one block per descriptor
__global__ void __launch_bounds__(128) naive_c2d_kernel(const C2dDesc* descs, char* base) {
  const C2dDesc d = descs[blockIdx.x];
  const uint32_t per_row = d.run_bytes >> 2, total = d.rows * per_row;
  for (uint32_t i = threadIdx.x; i < total; i += blockDim.x) {
    const uint32_t r = i / per_row, ch = i - r * per_row;
    *(uint32_t*)(base + d.dst_off + (int64_t)r * d.dst_stride + 4 * ch) =
        *(const uint32_t*)(base + d.src_off + (int64_t)r * d.src_stride + 4 * ch);
  }
}

int launch4(const Copy4& c, int n_sm, cudaStream_t st) {
  const uint64_t inner = (uint64_t)c.n[2] * c.run16, pairs = (uint64_t)c.n[0] * c.n[1];
  if (!inner || !pairs) return MOEBIUS_OK;
  if (inner >= (1ull << 31) || pairs > 65535) return MOEBIUS_E_INVAL;
  const uint64_t want = (inner + 4 * 256 - 1) / (4 * 256);
  const uint64_t per_pair = std::max<uint64_t>(1, ((uint64_t)n_sm * 16 + pairs - 1) / pairs);
  const dim3 grid((unsigned)std::min<uint64_t>(want, per_pair), (unsigned)pairs);
  naive_copy4d_kernel<<<grid, 256, 0, st>>>(c);
  return cudaGetLastError() == cudaSuccess ? MOEBIUS_OK : MOEBIUS_E_CUDA;
}

struct Need {
  int64_t w_bytes, kv_a, kv_b, desc_bytes, total;
};

// KV bookkeeping shared by the size query and the run: position of every page move inside its EP rank's
// packed list, pages per EP rank, prefix sums
struct KvIndex {
  std::vector<int32_t> pk;        // per move
  std::vector<int64_t> n_q, pre_q;
  int64_t total_pages = 0;
};

void kv_index(const moebius_plan_t* P, int R, KvIndex& ix) {
  ix.pk.assign((size_t)P->n_kv, 0);
  ix.n_q.assign((size_t)R, 0);
  ix.pre_q.assign((size_t)R + 1, 0);
  for (int64_t i = 0; i < P->n_kv; ++i) ix.pk[(size_t)i] = (int32_t)ix.n_q[(size_t)P->kv[i].ep_rank]++;
  for (int r = 0; r < R; ++r) ix.pre_q[(size_t)r + 1] = ix.pre_q[(size_t)r] + ix.n_q[(size_t)r];
  ix.total_pages = ix.pre_q[(size_t)R];
}

Need scratch_need(const moebius_ctx* x, const moebius_plan_t* P) {
  Need n;
  const int R = x->cfg.R;
  int max_slots = 0;
  for (int o = 0; o < x->n_obj; ++o) max_slots = std::max(max_slots, x->obj[o].n_slots);
  n.w_bytes = R > 1 ? (int64_t)R * x->S * max_slots : 0;
  const bool e2t = P->from == MOEBIUS_EP;
  n.kv_a = P->n_kv * x->ep_page_bytes;                                        // gathered, per-peer packed
  n.kv_b = e2t ? (int64_t)R * P->n_kv * x->tp_page_bytes : P->n_kv * x->ep_page_bytes;   // received
  // descriptor lists: gather (moves x groups), scatter (moves x receivers), exchange (R x R), scales
  n.desc_bytes = (P->n_kv * (int64_t)(x->G + std::max(x->G, R)) + (int64_t)R * R + 16) * (int64_t)sizeof(RowsDesc) +
                 (int64_t)P->c2d.size() * (int64_t)sizeof(C2dDesc) + 4096;
  n.total = std::max(n.w_bytes, n.kv_a + n.kv_b) + n.desc_bytes + 1024;
  return n;
}

}  // namespace
}  // namespace moebius

using namespace moebius;

extern "C" int moebius_naive_scratch_bytes(const moebius_ctx_t* x, const moebius_plan_t* P, int64_t* out) {
  if (!x || !P || !out || P->ctx != x) return MOEBIUS_E_INVAL;
  *out = (scratch_need(x, P).total + 255) / 256 * 256;
  return MOEBIUS_OK;
}

extern "C" int moebius_reshard_naive(moebius_ctx_t* x, const moebius_plan_t* P, void* dev_scratch, int64_t scratch_bytes,
                                     void* cuda_stream, int64_t* stats6) {
  if (!x || !P || P->ctx != x || !dev_scratch) return MOEBIUS_E_INVAL;
  if (!x->bound || x->active_mode != P->from) return MOEBIUS_E_STATE;
  if (!x->has_device || !x->prepared) return x->has_device ? MOEBIUS_E_STATE : MOEBIUS_E_CUDA;
  if (((uintptr_t)dev_scratch) & 255) return MOEBIUS_E_INVAL;
  const Need need = scratch_need(x, P);
  if (scratch_bytes < need.total) return MOEBIUS_E_INVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const moebius_config_t& c = x->cfg;
  const int R = c.R, L = c.L;
  const bool e2t = P->from == MOEBIUS_EP;
  char* base = x->base;
  char* buf = (char*)dev_scratch;                                   // staging: [weights A] or [KV A | KV B]
  char* dlist = buf + std::max(need.w_bytes, need.kv_a + need.kv_b);   // descriptor lists
  dlist = (char*)(((uintptr_t)dlist + 255) & ~(uintptr_t)255);
  int64_t bytes_read = 0, bytes_written = 0, launches = 0, w_passes_bytes = 0, kv_passes_bytes = 0;

  // ---- descriptor lists (host), uploaded before the timed launches ---------------------------------
  KvIndex ix;
  kv_index(P, R, ix);
  const int64_t run = x->run_kv;
  const int64_t tp_page = x->tp_page_bytes, ep_page = x->ep_page_bytes;
  std::vector<RowsDesc> gather, scatter, xchg;
  // Buffer A (sender side): EP->TP  rank q's chunk for group g:  [pre_q*G + g*n_q + pk][pg][run]
  //                         TP->EP  the chunk rank src(q,g) sends to q, same indexing by (q, g)
  // Buffer B (receiver):    EP->TP  rank j:  [j*total_pages + pre_q + pk][pg][run]
  //                         TP->EP  rank q:  [pre_q*G + g*n_q + pk][pg][run]   (== A's indexing)
  auto a_slot = [&](int q, int g, int32_t pk) { return (ix.pre_q[(size_t)q] * x->G + (int64_t)g * ix.n_q[(size_t)q] + pk) * tp_page; };
  for (int64_t i = 0; i < P->n_kv; ++i) {
    const KvDesc& d = P->kv[i];
    const uint32_t ntok = d.ntok_slot & 0xFFu;
    const int q = d.ep_rank;
    const int64_t ep_at = (int64_t)q * x->rank_stride + x->kv_off + (int64_t)d.ep_page * ep_page;
    for (int g = 0; g < x->G; ++g) {
      RowsDesc r;
      r.rows = ntok; r.run16 = (uint32_t)(run >> 4);
      if (e2t) {   // gather: EP page rows (stride G*run) of group g -> A
        r.a_off = ep_at + (int64_t)g * run; r.a_stride = (uint32_t)(x->G * run);
        r.b_off = a_slot(q, g, ix.pk[(size_t)i]); r.b_stride = (uint32_t)run;
        gather.push_back(r);
      } else {     // gather on the TP holder: TP page (contiguous rows) -> A ; scatter: B -> EP page rows
        const int j = (int)tp_src_rank((uint32_t)g, (uint32_t)x->rep, q);
        r.a_off = (int64_t)j * x->rank_stride + x->kv_off + (int64_t)d.tp_page * tp_page; r.a_stride = (uint32_t)run;
        r.b_off = a_slot(q, g, ix.pk[(size_t)i]); r.b_stride = (uint32_t)run;
        gather.push_back(r);
        RowsDesc s2 = r;
        s2.a_off = ep_at + (int64_t)g * run; s2.a_stride = (uint32_t)(x->G * run);
        scatter.push_back(s2);
      }
    }
    if (e2t) {
      for (int j = 0; j < R; ++j) {   // scatter on every TP rank: B_j -> TP page
        RowsDesc r;
        r.rows = ntok; r.run16 = (uint32_t)(run >> 4);
        r.a_off = (int64_t)j * x->rank_stride + x->kv_off + (int64_t)d.tp_page * tp_page; r.a_stride = (uint32_t)run;
        r.b_off = ((int64_t)j * ix.total_pages + ix.pre_q[(size_t)q] + ix.pk[(size_t)i]) * tp_page; r.b_stride = (uint32_t)run;
        scatter.push_back(r);
      }
    }
  }
  // exchange: whole chunks, A -> B (contiguous; expressed as 1-row descriptors of up to 2^32-1 chunks)
  for (int q = 0; q < R && P->n_kv; ++q) {
    const int64_t chunk = ix.n_q[(size_t)q] * tp_page;     // one group's packed pages of rank q
    if (!chunk) continue;
    if (e2t) {
      for (int g = 0; g < x->G; ++g)
        for (int rr = 0; rr < x->rep; ++rr) {
          const int j = g * x->rep + rr;
          RowsDesc r;
          r.rows = 1; r.run16 = (uint32_t)(chunk >> 4); r.a_stride = r.b_stride = 0;
          r.a_off = a_slot(q, g, 0);
          r.b_off = ((int64_t)j * ix.total_pages + ix.pre_q[(size_t)q]) * tp_page;
          xchg.push_back(r);
        }
    } else {
      for (int g = 0; g < x->G; ++g) {
        RowsDesc r;
        r.rows = 1; r.run16 = (uint32_t)(chunk >> 4); r.a_stride = r.b_stride = 0;
        r.a_off = a_slot(q, g, 0); r.b_off = a_slot(q, g, 0);
        xchg.push_back(r);
      }
    }
  }
  char* d_gather = dlist;
  char* d_scatter = d_gather + gather.size() * sizeof(RowsDesc);
  char* d_xchg = d_scatter + scatter.size() * sizeof(RowsDesc);
  char* d_c2d = d_xchg + xchg.size() * sizeof(RowsDesc);
  if (d_c2d + P->c2d.size() * sizeof(C2dDesc) > buf + scratch_bytes) return MOEBIUS_E_INVAL;
  auto up = [&](char* dst, const void* src, size_t n) { return !n || cudaMemcpyAsync(dst, src, n, cudaMemcpyHostToDevice, st) == cudaSuccess; };
  if (!up(d_gather, gather.data(), gather.size() * sizeof(RowsDesc)) || !up(d_scatter, scatter.data(), scatter.size() * sizeof(RowsDesc)) ||
      !up(d_xchg, xchg.data(), xchg.size() * sizeof(RowsDesc)) || !up(d_c2d, P->c2d.data(), P->c2d.size() * sizeof(C2dDesc)))
    return MOEBIUS_E_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return MOEBIUS_E_CUDA;   // the host vectors die with this call

  cudaEvent_t ev_a = nullptr, ev_b = nullptr;
  if (x->timing) {
    int64_t k = x->ev_count % kTimingRing;
    ev_a = (cudaEvent_t)x->ev[2 * k]; ev_b = (cudaEvent_t)x->ev[2 * k + 1];
    cudaEventRecord(ev_a, st);
  }

  // ---- expert weights: per (layer, matrix) object in the direction-specific chain order -------------
  if (R > 1) {
    const int n_links = L * x->n_obj;
    for (int step = 0; step < n_links; ++step) {
      const int k = e2t ? step : n_links - 1 - step;
      const int layer = k / x->n_obj;
      const WObj& ob = x->obj[k % x->n_obj];
      const int tp_slot = 3 * layer + ob.slot;
      const int64_t runb = !ob.long_run ? (int64_t)(c.I / R) * x->wb : (int64_t)(c.I / R) * c.H * x->wb;
      const int64_t rows = !ob.long_run ? (int64_t)(c.E / R) * c.H : (int64_t)(c.E / R) * ob.row_mult;
      const int64_t obj_bytes = rows * R * runb;                 // one rank's view (n_slots * S up to padding)
      char* tp0 = base + x->w_off + (int64_t)tp_slot * x->S;
      char* ep0 = base + x->w_off + (int64_t)(tp_slot + x->ep_shift) * x->S;
      Copy4 perm, exch;
      // permute: EP view [rows][R][run]  <->  buffer A_q = [j][rows][run]
      perm.n[0] = (uint32_t)R; perm.n[1] = (uint32_t)R; perm.n[2] = (uint32_t)rows; perm.run16 = (uint32_t)(runb >> 4);
      const int64_t ep_s[3] = {x->rank_stride, runb, R * runb}, a_s[3] = {obj_bytes, rows * runb, runb};
      // exchange: chunk (q, j) of A  <->  block q of rank j's TP view; rows*run contiguous bytes each
      const int64_t piece16 = (rows * runb) >> 4;
      const uint32_t split = (uint32_t)((piece16 + (1u << 30) - 1) >> 30);   // keep run16 below 2^32
      exch.n[0] = (uint32_t)R; exch.n[1] = (uint32_t)R; exch.n[2] = split; exch.run16 = (uint32_t)(piece16 / split);
      if (piece16 % split) return MOEBIUS_E_INVAL;
      const int64_t sub = (piece16 / split) << 4;
      const int64_t xa_s[3] = {obj_bytes, rows * runb, sub}, tp_s[3] = {rows * runb, x->rank_stride, sub};
      if (e2t) {
        perm.src = ep0; perm.dst = buf; memcpy(perm.ss, ep_s, sizeof(ep_s)); memcpy(perm.ds, a_s, sizeof(a_s));
        exch.src = buf; exch.dst = tp0; memcpy(exch.ss, xa_s, sizeof(xa_s)); memcpy(exch.ds, tp_s, sizeof(tp_s));
        if (int rc = launch4(perm, x->n_sm, st)) return rc;
        if (int rc = launch4(exch, x->n_sm, st)) return rc;
      } else {
        exch.src = tp0; exch.dst = buf; memcpy(exch.ss, tp_s, sizeof(tp_s)); memcpy(exch.ds, xa_s, sizeof(xa_s));
        perm.src = buf; perm.dst = ep0; memcpy(perm.ss, a_s, sizeof(a_s)); memcpy(perm.ds, ep_s, sizeof(ep_s));
        if (int rc = launch4(exch, x->n_sm, st)) return rc;
        if (int rc = launch4(perm, x->n_sm, st)) return rc;
      }
      launches += 2;
      w_passes_bytes += 2 * obj_bytes * R;
    }
    bytes_read += w_passes_bytes; bytes_written += w_passes_bytes;
  }
  // fp8 block scales: disjoint fixed regions, one direct pass (2.4 MB at config 5)
  if (!P->c2d.empty()) {
    naive_c2d_kernel<<<(unsigned)P->c2d.size(), 128, 0, st>>>((const C2dDesc*)d_c2d, base);
    if (cudaGetLastError() != cudaSuccess) return MOEBIUS_E_CUDA;
    ++launches;
  }
  // attention head shards (memory-saving variant): an All-Gather is already one pass per element
  for (size_t i = 0; i < P->segs.size(); ++i) {
    const Seg& s = P->segs[i];
    if (seg_kind(s) != SEG_BULK) continue;
    for (uint32_t di = 0; di < s.n_desc; ++di) {
      const BulkDesc& d = P->bulk[s.desc_begin + di];
      Copy4 cp;
      cp.src = base + d.src_off; cp.dst = base + d.dst_off;
      cp.n[0] = 1; cp.n[1] = 1; cp.n[2] = s.rows_total; cp.run16 = (uint32_t)(((int64_t)s.chunk_bytes * s.chunks_per_run) >> 4);
      cp.ss[0] = cp.ss[1] = cp.ds[0] = cp.ds[1] = 0; cp.ss[2] = s.ep_off; cp.ds[2] = s.tp_off;
      if (int rc = launch4(cp, x->n_sm, st)) return rc;
      ++launches;
    }
  }
  // ---- paged KV: per pool gather -> exchange -> scatter ------------------------------------------------
  if (P->n_kv) {
    char* A = buf;
    char* B = buf + need.kv_a;
    const unsigned ysplit = 2;
    for (int z = 0; z < 2 * L; ++z) {
      char* pool = base + (int64_t)z * x->pool_bytes;      // descriptors carry rank + kv_off + page offsets
      naive_rows_kernel<<<dim3((unsigned)gather.size(), ysplit), 128, 0, st>>>((const RowsDesc*)d_gather, pool, A, 1);
      naive_rows_kernel<<<dim3((unsigned)xchg.size(), 512), 128, 0, st>>>((const RowsDesc*)d_xchg, A, B, 1);
      naive_rows_kernel<<<dim3((unsigned)scatter.size(), ysplit), 128, 0, st>>>((const RowsDesc*)d_scatter, pool, B, 0);
      if (cudaGetLastError() != cudaSuccess) return MOEBIUS_E_CUDA;
      launches += 3;
    }
    const int64_t rd = P->stats.kv_read, wr = P->stats.kv_relocated;
    // gather reads the source once and writes it packed; exchange reads it and writes every receiver's
    // copy; scatter reads those and writes the target pages
    kv_passes_bytes = (rd + rd) + (rd + wr) + (wr + wr);
    bytes_read += rd + rd + wr; bytes_written += rd + wr + wr;
  }
  if (x->timing) { cudaEventRecord(ev_b, st); x->ev_count++; }
  // publish, as moebius_reshard does
  if (cudaMemcpyAsync(x->tables, P->tbl_image, (size_t)P->tbl_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return MOEBIUS_E_CUDA;
  if (P->buf.ev && cudaEventRecord((cudaEvent_t)P->buf.ev, st) != cudaSuccess) return MOEBIUS_E_CUDA;
  x->active_mode = P->to;
  x->switch_count++;
  if (stats6) {
    stats6[0] = launches; stats6[1] = bytes_read; stats6[2] = bytes_written;
    stats6[3] = w_passes_bytes; stats6[4] = kv_passes_bytes; stats6[5] = need.total;
  }
  return MOEBIUS_OK;
}
