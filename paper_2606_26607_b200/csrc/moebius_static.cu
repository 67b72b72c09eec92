// moebius_static.cu -- the staged comparison path with its scratch in a STATIC device array.
//
// moebius_reshard_naive (moebius_naive.cu; Table 1 :176-189) needs a caller-owned
// staging buffer.  Some callers cannot provide one because they cannot call cudaMalloc where they stand
// (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  This file gives them
// ONE entry point that allocates no device memory: the same kernels, the same plan, the same result bit
// for bit, with the staging buffer in the file-scope array below.
//
//  * The array is MOEBIUS_STATIC_SCRATCH_BYTES (64 MiB) of device memory per GPU that loads this library,
//    held until the process exits.  A plan that needs more is refused (MOEBIUS_E_STAGING).
//  * In HOST code the array's name is a host-side stand-in, not a device address: a kernel given it
//    faults, or reads the wrong memory.  The device address comes from cudaGetSymbolAddress, asked once
//    per device with that device current (device_scratch below), and that pointer is what the kernels get.
//  * Every call shares the array, which keeps the previous call's bytes.  Nothing in it has to start at
//    zero: each launch of the staged path reads only what an earlier launch of the SAME call wrote
//    (permute -> exchange, gather -> exchange -> scatter), so nothing is cleared.  Two calls that overlap
//    on the GPU (different streams, different contexts on one device) race on it: serialise them.
#include <cuda_runtime.h>

#include <mutex>

#include "moebius_host.h"

namespace {

constexpr int64_t kStaticScratchBytes = (int64_t)MOEBIUS_STATIC_SCRATCH_BYTES;
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned char g_static_scratch[MOEBIUS_STATIC_SCRATCH_BYTES];

std::mutex g_mu;
void* g_ptr[kMaxDevices];      // device address of g_static_scratch on device d (nullptr: not asked yet)

// The device address of the array on the CURRENT device.  cudaGetSymbolAddress is called once per device.
int device_scratch(void** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return MOEBIUS_E_CUDA; }
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_ptr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) { cudaGetLastError(); return MOEBIUS_E_CUDA; }
    if (((uintptr_t)p) & 255) return MOEBIUS_E_CUDA;
    g_ptr[dev] = p;
  }
  *out = g_ptr[dev];
  return MOEBIUS_OK;
}

}  // namespace

extern "C" int64_t moebius_static_scratch_bytes(void) { return kStaticScratchBytes; }

extern "C" int moebius_reshard_naive_static(moebius_ctx_t* x, const moebius_plan_t* P, void* cuda_stream, int64_t* stats6) {
  if (!x || !P) return MOEBIUS_E_INVAL;
  int64_t need = 0;
  if (int rc = moebius_naive_scratch_bytes(x, P, &need)) return rc;
  if (need > kStaticScratchBytes) return MOEBIUS_E_STAGING;      // "staging buffer too small": the limit is fixed
  void* scratch = nullptr;
  if (int rc = device_scratch(&scratch)) return rc;
  // the kernels of the staged path, handed the array's DEVICE address
  return moebius_reshard_naive(x, P, scratch, kStaticScratchBytes, cuda_stream, stats6);
}
