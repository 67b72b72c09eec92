// moebius_arena.cu -- the unified buffer as ONE virtual address range over SEPARATE physical
// allocations, one per rank (CUDA virtual memory management).
//
// every rank's buffer has a fixed address, is exported once (CUDA IPC) and mapped
// by its peers, and the transfer kernels store into the peers' slots.  The B200-native form of that:
// reserve R * rank_stride bytes of virtual address space, back rank r's region with its own physical
// allocation (on this GPU, or imported from the process that owns rank r through a POSIX file
// descriptor), and map it at base + r * rank_stride.  Every address the planner and the kernel
// compute -- including the tensor maps, whose rank dimension has stride rank_stride -- is then valid
// unchanged whether the ranks are regions of one GPU or one GPU each.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstring>
#include <new>
#include <vector>

#include "moebius_host.h"

namespace {

struct Driver {
  CUresult (*AddressReserve)(CUdeviceptr*, size_t, size_t, CUdeviceptr, unsigned long long);
  CUresult (*AddressFree)(CUdeviceptr, size_t);
  CUresult (*Create)(CUmemGenericAllocationHandle*, size_t, const CUmemAllocationProp*, unsigned long long);
  CUresult (*Release)(CUmemGenericAllocationHandle);
  CUresult (*Map)(CUdeviceptr, size_t, size_t, CUmemGenericAllocationHandle, unsigned long long);
  CUresult (*Unmap)(CUdeviceptr, size_t);
  CUresult (*SetAccess)(CUdeviceptr, size_t, const CUmemAccessDesc*, size_t);
  CUresult (*Granularity)(size_t*, const CUmemAllocationProp*, CUmemAllocationGranularity_flags);
  CUresult (*Export)(void*, CUmemGenericAllocationHandle, CUmemAllocationHandleType, unsigned long long);
  CUresult (*Import)(CUmemGenericAllocationHandle*, void*, CUmemAllocationHandleType);
  bool ok;
};

template <typename F>
bool entry(const char* name, F* out) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint(name, &fn, cudaEnableDefault, &q) != cudaSuccess || !fn) {
    cudaGetLastError();
    return false;
  }
  *out = (F)fn;
  return true;
}

bool load_driver(Driver* d) {
  d->ok = entry("cuMemAddressReserve", &d->AddressReserve) && entry("cuMemAddressFree", &d->AddressFree) &&
          entry("cuMemCreate", &d->Create) && entry("cuMemRelease", &d->Release) && entry("cuMemMap", &d->Map) &&
          entry("cuMemUnmap", &d->Unmap) && entry("cuMemSetAccess", &d->SetAccess) &&
          entry("cuMemGetAllocationGranularity", &d->Granularity) &&
          entry("cuMemExportToShareableHandle", &d->Export) && entry("cuMemImportFromShareableHandle", &d->Import);
  return d->ok;
}

}  // namespace

struct moebius_arena {
  Driver drv;
  int device;
  int R;
  int64_t rank_stride;
  CUdeviceptr va;
  std::vector<CUmemGenericAllocationHandle> handle;   // per rank; 0 = not mapped yet
  std::vector<uint8_t> mapped, local;
};

extern "C" {

int moebius_arena_create(const moebius_ctx_t* x, int device, int rank_lo, int rank_hi, moebius_arena_t** out) {
  if (!x || !out) return MOEBIUS_E_INVAL;
  *out = nullptr;
  const int R = x->cfg.R;
  if (rank_lo < 0 || rank_hi > R || rank_lo > rank_hi) return MOEBIUS_E_INVAL;
  if (cudaSetDevice(device) != cudaSuccess || cudaFree(nullptr) != cudaSuccess) { cudaGetLastError(); return MOEBIUS_E_CUDA; }
  moebius_arena* a = new (std::nothrow) moebius_arena();
  if (!a) return MOEBIUS_E_INVAL;
  if (!load_driver(&a->drv)) { delete a; return MOEBIUS_E_CUDA; }
  a->device = device; a->R = R; a->rank_stride = x->rank_stride; a->va = 0;
  a->handle.assign((size_t)R, 0); a->mapped.assign((size_t)R, 0); a->local.assign((size_t)R, 0);
  CUmemAllocationProp prop;
  memset(&prop, 0, sizeof(prop));
  prop.type = CU_MEM_ALLOCATION_TYPE_PINNED;
  prop.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
  prop.location.id = device;
  prop.requestedHandleTypes = CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR;
  size_t gran = 0;
  if (a->drv.Granularity(&gran, &prop, CU_MEM_ALLOC_GRANULARITY_MINIMUM) != CUDA_SUCCESS || gran == 0 ||
      a->rank_stride % (int64_t)gran) {
    delete a;
    return MOEBIUS_E_INVAL;   // rank_stride is a multiple of 2 MiB; a coarser granularity is not supported
  }
  if (a->drv.AddressReserve(&a->va, (size_t)(a->rank_stride * R), (size_t)gran, 0, 0) != CUDA_SUCCESS) {
    delete a;
    return MOEBIUS_E_CUDA;
  }
  CUmemAccessDesc acc;
  memset(&acc, 0, sizeof(acc));
  acc.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
  acc.location.id = device;
  acc.flags = CU_MEM_ACCESS_FLAGS_PROT_READWRITE;
  for (int r = rank_lo; r < rank_hi; ++r) {
    CUdeviceptr at = a->va + (CUdeviceptr)((int64_t)r * a->rank_stride);
    if (a->drv.Create(&a->handle[(size_t)r], (size_t)a->rank_stride, &prop, 0) != CUDA_SUCCESS ||
        a->drv.Map(at, (size_t)a->rank_stride, 0, a->handle[(size_t)r], 0) != CUDA_SUCCESS) {
      moebius_arena_destroy(a);
      return MOEBIUS_E_CUDA;
    }
    a->mapped[(size_t)r] = 1;   // mapped from here on: destroy must unmap it even if SetAccess fails
    a->local[(size_t)r] = 1;
    if (a->drv.SetAccess(at, (size_t)a->rank_stride, &acc, 1) != CUDA_SUCCESS) {
      moebius_arena_destroy(a);
      return MOEBIUS_E_CUDA;
    }
  }
  *out = a;
  return MOEBIUS_OK;
}

void moebius_arena_destroy(moebius_arena_t* a) {
  if (!a) return;
  for (int r = 0; r < a->R; ++r) {
    CUdeviceptr at = a->va + (CUdeviceptr)((int64_t)r * a->rank_stride);
    if (a->mapped[(size_t)r]) a->drv.Unmap(at, (size_t)a->rank_stride);
    if (a->handle[(size_t)r]) a->drv.Release(a->handle[(size_t)r]);
  }
  if (a->va) a->drv.AddressFree(a->va, (size_t)(a->rank_stride * a->R));
  delete a;
}

void* moebius_arena_base(const moebius_arena_t* a) { return a ? (void*)a->va : nullptr; }

int moebius_arena_ready(const moebius_arena_t* a) {
  if (!a) return MOEBIUS_E_INVAL;
  for (int r = 0; r < a->R; ++r) if (!a->mapped[(size_t)r]) return MOEBIUS_E_STATE;
  return MOEBIUS_OK;
}

int moebius_arena_export(const moebius_arena_t* a, int rank, int* fd_out) {
  if (!a || !fd_out || rank < 0 || rank >= a->R) return MOEBIUS_E_INVAL;
  if (!a->local[(size_t)rank]) return MOEBIUS_E_STATE;
  int fd = -1;
  if (a->drv.Export(&fd, a->handle[(size_t)rank], CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR, 0) != CUDA_SUCCESS)
    return MOEBIUS_E_CUDA;
  *fd_out = fd;
  return MOEBIUS_OK;
}

int moebius_arena_import(moebius_arena_t* a, int rank, int fd) {
  if (!a || rank < 0 || rank >= a->R || fd < 0) return MOEBIUS_E_INVAL;
  if (a->mapped[(size_t)rank]) return MOEBIUS_E_STATE;
  CUmemGenericAllocationHandle h = 0;
  if (a->drv.Import(&h, (void*)(uintptr_t)fd, CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR) != CUDA_SUCCESS)
    return MOEBIUS_E_CUDA;
  CUdeviceptr at = a->va + (CUdeviceptr)((int64_t)rank * a->rank_stride);
  CUmemAccessDesc acc;
  memset(&acc, 0, sizeof(acc));
  acc.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
  acc.location.id = a->device;
  acc.flags = CU_MEM_ACCESS_FLAGS_PROT_READWRITE;
  if (a->drv.Map(at, (size_t)a->rank_stride, 0, h, 0) != CUDA_SUCCESS) { a->drv.Release(h); return MOEBIUS_E_CUDA; }
  if (a->drv.SetAccess(at, (size_t)a->rank_stride, &acc, 1) != CUDA_SUCCESS) {
    a->drv.Unmap(at, (size_t)a->rank_stride);
    a->drv.Release(h);
    return MOEBIUS_E_CUDA;
  }
  a->handle[(size_t)rank] = h;
  a->mapped[(size_t)rank] = 1;
  return MOEBIUS_OK;
}

}  // extern "C"
