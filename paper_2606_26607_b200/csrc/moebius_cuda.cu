// moebius_cuda.cu -- the fused reshard kernel for sm_100a and its launch path.
//
// ONE persistent kernel executes the whole work list of a switch (expert-weight slices, KV pages,
// staging copies, scale copies): "reads from the source-mode alias and writes the slice
// into the ... target-mode slot" -- one HBM read and one write per element (Table 1).
// The paper's H200 kernels push slices over NVLink to peers; here the R ranks are regions of one
// allocation, so the same descriptors drive an on-device relayout bounded by HBM bandwidth.
//
// Scheduling: each warp takes unit ids from one global ticket, in list order; a unit is <= ~32 KB.
// Data path: 16-byte ld.global / st.global with L1 no-allocate, 8 loads in flight per lane, lanes
// mapped to consecutive 16-byte chunks of the EP-side row so that both sides are accessed in whole
// contiguous runs (>= one 32-byte sector, usually whole 128-byte lines).
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

__global__ void __launch_bounds__(512, 1) moebius_reshard_kernel(const DevParams p) {
  const uint32_t lane = threadIdx.x & 31;
  uint32_t si = 0;
  for (;;) {
    uint32_t u = 0;
    if (lane == 0) u = atomicAdd(p.ticket, 1u);
    u = __shfl_sync(0xffffffffu, u, 0);
    if (u >= p.total_units) break;
    // units are handed out in increasing order: search forward from the last segment
    while (si + 1 < p.n_segs && u >= __ldg(&p.segs[si + 1].unit_begin)) {
      uint32_t lo = si + 1, hi = p.n_segs - 1;  // last segment whose unit_begin <= u
      while (lo < hi) {
        uint32_t mid = (lo + hi + 1) >> 1;
        if (__ldg(&p.segs[mid].unit_begin) <= u) lo = mid; else hi = mid - 1;
      }
      si = lo;
    }
    const Seg s = p.segs[si];
    const uint32_t ul = u - s.unit_begin;
    if (s.wait_ctr >= 0) {
      if (lane == 0) {
        const uint32_t* c = p.counters + s.wait_ctr;
        while (ld_acquire(c) < s.wait_target) __nanosleep(200);
      }
      __syncwarp();
    }
    if (s.kind == SEG_COPY2D) {
      c2d_copy(p.c2d[s.desc_begin + ul], p.base, lane);
    } else {
      const uint32_t nb = seg_boxes(s, ul);
      for (uint32_t k = 0; k < nb; ++k) {
        Box b;
        decode_box(s, p, ul, k, b);
        if (b.lin) lin_copy(b.lin_src, b.lin_dst, b.lin_bytes, lane);
        else if (s.ep_is_src) xbox_ep_to_tp(b, p.rank_stride, lane);
        else xbox_tp_to_ep(b, p.rank_stride, lane);
      }
    }
    if (s.signal_ctr >= 0) {
      __syncwarp();
      if (lane == 0) {
        __threadfence();
        atomicAdd(p.counters + s.signal_ctr, 1u);
      }
    }
  }
}

void* host_alloc(int64_t bytes, bool* pinned) {
  void* p = nullptr;
  *pinned = false;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) == cudaSuccess && ndev > 0 &&
      cudaHostAlloc(&p, (size_t)bytes, cudaHostAllocDefault) == cudaSuccess) {
    *pinned = true;
    return p;
  }
  cudaGetLastError();
  return malloc((size_t)bytes);
}

void host_free(void* p, bool pinned) {
  if (!p) return;
  if (pinned) cudaFreeHost(p); else free(p);
}

void cuda_ctx_destroy(moebius_ctx* x) {
  if (x->ev_valid) {
    for (int i = 0; i < 2 * kTimingRing; ++i) cudaEventDestroy((cudaEvent_t)x->ev[i]);
    x->ev_valid = false;
  }
}

}  // namespace moebius

using namespace moebius;

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
  return MOEBIUS_OK;
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

extern "C" int moebius_reshard(moebius_ctx_t* x, const moebius_plan_t* P, void* cuda_stream) {
  if (!x || !P || P->ctx != x) return MOEBIUS_E_INVAL;
  if (!x->bound || x->active_mode != P->from) return MOEBIUS_E_STATE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (x->n_sm == 0) {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return MOEBIUS_E_CUDA;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return MOEBIUS_E_CUDA;
    x->n_sm = n;
  }
  if (x->timing && !x->ev_valid) {
    for (int i = 0; i < 2 * kTimingRing; ++i) {
      cudaEvent_t e;
      if (cudaEventCreate(&e) != cudaSuccess) return MOEBIUS_E_CUDA;
      x->ev[i] = e;
    }
    x->ev_valid = true;
  }
  cudaEvent_t ev_a = nullptr, ev_b = nullptr;
  if (x->timing) {
    int64_t k = x->ev_count % kTimingRing;
    ev_a = (cudaEvent_t)x->ev[2 * k]; ev_b = (cudaEvent_t)x->ev[2 * k + 1];
  }
  // 1. work list -> device; ticket and the counters this plan uses -> 0
  if (cudaMemsetAsync(x->desc, 0, (size_t)(kCtrOff + 4 * (int64_t)(P->n_counters ? P->n_counters : 1)), st) != cudaSuccess)
    return MOEBIUS_E_CUDA;
  if (P->image_bytes &&
      cudaMemcpyAsync(x->desc + kSegOff, P->image, (size_t)P->image_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess)
    return MOEBIUS_E_CUDA;
  // 2. the kernel
  if (P->total_units) {
    DevParams p;
    p.base = x->base;
    p.stg = x->stg;
    p.segs = (const Seg*)(x->desc + kSegOff);
    p.kv = (const KvDesc*)(x->desc + kSegOff + P->kv_img_off);
    p.c2d = (const C2dDesc*)(x->desc + kSegOff + P->c2d_img_off);
    p.ticket = (uint32_t*)x->desc;
    p.counters = (uint32_t*)(x->desc + kCtrOff);
    p.rank_stride = x->rank_stride;
    p.n_segs = (uint32_t)P->segs.size();
    p.total_units = P->total_units;
    int threads = x->threads > 0 ? x->threads : 512;
    int per_sm = x->ctas_per_sm > 0 ? x->ctas_per_sm : 2;
    int64_t warps_needed = P->total_units;
    int64_t grid = (int64_t)x->n_sm * per_sm;
    int64_t grid_cap = (warps_needed + threads / 32 - 1) / (threads / 32);
    if (grid > grid_cap) grid = grid_cap;
    if (x->timing) cudaEventRecord(ev_a, st);
    moebius_reshard_kernel<<<(unsigned)grid, threads, 0, st>>>(p);
    if (cudaGetLastError() != cudaSuccess) return MOEBIUS_E_CUDA;
    if (x->timing) cudaEventRecord(ev_b, st);
  } else if (x->timing) {
    cudaEventRecord(ev_a, st);
    cudaEventRecord(ev_b, st);
  }
  if (x->timing) x->ev_count++;
  // 3. publish: new tables, owner vector and the active-mode flag at their fixed address
  if (cudaMemcpyAsync(x->tables, P->tbl_image, (size_t)P->tbl_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess)
    return MOEBIUS_E_CUDA;
  x->active_mode = P->to;
  x->switch_count++;
  return MOEBIUS_OK;
}
