// NEXT-3: a dW accumulator STITCHED from per-rank shards with CUDA virtual memory
// management, so that the A6 epilogue's TMA reduce-add IS the data-parallel reduce-scatter.
//
// Every rank creates one physical chunk on its own GPU (cuMemCreate, exportable as a POSIX file descriptor), the
// ranks exchange the descriptors, and every rank maps ALL chunks, in rank order, into one contiguous virtual range
// (cuMemAddressReserve + cuMemMap + cuMemSetAccess): rows [r R, (r+1) R) of the fp32 [V, d] gradient physically
// live on rank r.  Handed to grpo_fused_logprob_loss_bwd / grpo_enqueue_groups as `dW_accum`, that range needs no
// kernel change: the contraction kernel's epilogue already issues element-wise fp32 reduce-adds
// (cp.reduce.async.bulk.tensor ... .add, performed at the L2 of the memory's home GPU), which NVLink carries to a
// peer's HBM like any other store.  All ranks add their tiles into every shard while their GEMMs run; after a
// barrier each rank holds the fully reduced rows of its shard - GEMM -> reduce-scatter in ONE kernel, the transfer
// overlapped with the math tile by tile, no all-reduce afterwards (a sharded optimizer step and an all-gather of
// the updated weights follow, as with any ZeRO-1 style data parallelism).
//
// Host code only; driver entry points are resolved at run time (no link against libcuda).
#include "../../include/grpo.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <map>
#include <mutex>
#include <new>
#include <vector>

int32_t grpo_internal_fail(int32_t code, const char* fmt, ...);   // grpo_api.cu: sets grpo_last_error()

struct grpo_shard {
  CUmemGenericAllocationHandle handle;
  size_t bytes;
};

namespace {
struct Vmm {
  CUresult (*GetGranularity)(size_t*, const CUmemAllocationProp*, CUmemAllocationGranularity_flags) = nullptr;
  CUresult (*Create)(CUmemGenericAllocationHandle*, size_t, const CUmemAllocationProp*, unsigned long long) = nullptr;
  CUresult (*Release)(CUmemGenericAllocationHandle) = nullptr;
  CUresult (*Export)(void*, CUmemGenericAllocationHandle, CUmemAllocationHandleType, unsigned long long) = nullptr;
  CUresult (*Import)(CUmemGenericAllocationHandle*, void*, CUmemAllocationHandleType) = nullptr;
  CUresult (*Reserve)(CUdeviceptr*, size_t, size_t, CUdeviceptr, unsigned long long) = nullptr;
  CUresult (*AddressFree)(CUdeviceptr, size_t) = nullptr;
  CUresult (*Map)(CUdeviceptr, size_t, size_t, CUmemGenericAllocationHandle, unsigned long long) = nullptr;
  CUresult (*Unmap)(CUdeviceptr, size_t) = nullptr;
  CUresult (*SetAccess)(CUdeviceptr, size_t, const CUmemAccessDesc*, size_t) = nullptr;
  bool ok = false;
};

template <typename F>
bool resolve(const char* name, F& fn) {
  void* p = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint(name, &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess || !p)
    return false;
  fn = reinterpret_cast<F>(p);
  return true;
}

const Vmm& vmm() {
  static Vmm v;
  static std::once_flag once;
  std::call_once(once, [] {
    v.ok = resolve("cuMemGetAllocationGranularity", v.GetGranularity) && resolve("cuMemCreate", v.Create) &&
           resolve("cuMemRelease", v.Release) && resolve("cuMemExportToShareableHandle", v.Export) &&
           resolve("cuMemImportFromShareableHandle", v.Import) && resolve("cuMemAddressReserve", v.Reserve) &&
           resolve("cuMemAddressFree", v.AddressFree) && resolve("cuMemMap", v.Map) && resolve("cuMemUnmap", v.Unmap) &&
           resolve("cuMemSetAccess", v.SetAccess);
  });
  return v;
}

CUmemAllocationProp shard_prop(int device) {
  CUmemAllocationProp prop = {};
  prop.type = CU_MEM_ALLOCATION_TYPE_PINNED;
  prop.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
  prop.location.id = device;
  prop.requestedHandleTypes = CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR;
  return prop;
}

std::mutex g_mu;
std::map<void*, size_t> g_ranges;   // stitched ranges: base -> total bytes

int current_device(int* dev) { return cudaGetDevice(dev) == cudaSuccess ? 0 : -1; }
}  // namespace

#define VMM_OK(expr)                                                                                         \
  do {                                                                                                       \
    CUresult r__ = (expr);                                                                                   \
    if (r__ != CUDA_SUCCESS) return grpo_internal_fail(GRPO_ERR_CUDA, "%s failed with CUresult %d", #expr, (int)r__); \
  } while (0)

extern "C" int32_t grpo_shard_granularity(grpo_ctx* ctx, int64_t* bytes_out) {
  if (!ctx || !bytes_out) return grpo_internal_fail(GRPO_ERR_INVALID_ARG, "ctx / bytes_out is NULL");
  if (!vmm().ok) return grpo_internal_fail(GRPO_ERR_CUDA, "CUDA virtual memory management entry points not available");
  int dev = 0;
  if (current_device(&dev)) return grpo_internal_fail(GRPO_ERR_CUDA, "cudaGetDevice failed");
  const CUmemAllocationProp prop = shard_prop(dev);
  size_t g = 0;
  VMM_OK(vmm().GetGranularity(&g, &prop, CU_MEM_ALLOC_GRANULARITY_RECOMMENDED));
  *bytes_out = static_cast<int64_t>(g);
  return GRPO_OK;
}

extern "C" int32_t grpo_shard_create(grpo_ctx* ctx, int64_t bytes, grpo_shard** shard_out, int32_t* fd_out) {
  if (!ctx || !shard_out || bytes <= 0) return grpo_internal_fail(GRPO_ERR_INVALID_ARG, "bad ctx / shard_out / bytes");
  int64_t gran = 0;
  int32_t st = grpo_shard_granularity(ctx, &gran);
  if (st != GRPO_OK) return st;
  if (bytes % gran != 0)
    return grpo_internal_fail(GRPO_ERR_SHAPE, "shard bytes %lld is not a multiple of the allocation granularity %lld",
                              (long long)bytes, (long long)gran);
  int dev = 0;
  if (current_device(&dev)) return grpo_internal_fail(GRPO_ERR_CUDA, "cudaGetDevice failed");
  const CUmemAllocationProp prop = shard_prop(dev);
  grpo_shard* s = new (std::nothrow) grpo_shard();
  if (!s) return grpo_internal_fail(GRPO_ERR_INVALID_ARG, "out of host memory");
  s->bytes = static_cast<size_t>(bytes);
  CUresult r = vmm().Create(&s->handle, s->bytes, &prop, 0);
  if (r != CUDA_SUCCESS) {
    delete s;
    return grpo_internal_fail(GRPO_ERR_CUDA, "cuMemCreate(%lld bytes) failed with CUresult %d", (long long)bytes, (int)r);
  }
  if (fd_out) {
    int fd = -1;
    r = vmm().Export(&fd, s->handle, CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR, 0);
    if (r != CUDA_SUCCESS) {
      vmm().Release(s->handle);
      delete s;
      return grpo_internal_fail(GRPO_ERR_CUDA, "cuMemExportToShareableHandle failed with CUresult %d", (int)r);
    }
    *fd_out = fd;
  }
  *shard_out = s;
  return GRPO_OK;
}

extern "C" int32_t grpo_shard_import(grpo_ctx* ctx, int32_t fd, int64_t bytes, grpo_shard** shard_out) {
  if (!ctx || !shard_out || fd < 0 || bytes <= 0) return grpo_internal_fail(GRPO_ERR_INVALID_ARG, "bad ctx / fd / bytes");
  if (!vmm().ok) return grpo_internal_fail(GRPO_ERR_CUDA, "CUDA virtual memory management entry points not available");
  grpo_shard* s = new (std::nothrow) grpo_shard();
  if (!s) return grpo_internal_fail(GRPO_ERR_INVALID_ARG, "out of host memory");
  s->bytes = static_cast<size_t>(bytes);
  CUresult r = vmm().Import(&s->handle, reinterpret_cast<void*>(static_cast<uintptr_t>(fd)),
                            CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR);
  if (r != CUDA_SUCCESS) {
    delete s;
    return grpo_internal_fail(GRPO_ERR_CUDA, "cuMemImportFromShareableHandle failed with CUresult %d", (int)r);
  }
  *shard_out = s;
  return GRPO_OK;
}

extern "C" int32_t grpo_shard_release(grpo_ctx* ctx, grpo_shard* shard) {
  if (!ctx) return grpo_internal_fail(GRPO_ERR_INVALID_ARG, "ctx is NULL");
  if (!shard) return GRPO_OK;
  const CUresult r = vmm().ok ? vmm().Release(shard->handle) : CUDA_SUCCESS;
  delete shard;
  if (r != CUDA_SUCCESS) return grpo_internal_fail(GRPO_ERR_CUDA, "cuMemRelease failed with CUresult %d", (int)r);
  return GRPO_OK;
}

extern "C" int32_t grpo_stitch_map(grpo_ctx* ctx, grpo_shard* const* shards, int32_t n, void** dev_ptr_out) {
  if (!ctx || !shards || n < 1 || !dev_ptr_out) return grpo_internal_fail(GRPO_ERR_INVALID_ARG, "bad arguments");
  if (!vmm().ok) return grpo_internal_fail(GRPO_ERR_CUDA, "CUDA virtual memory management entry points not available");
  size_t total = 0;
  for (int i = 0; i < n; ++i) {
    if (!shards[i]) return grpo_internal_fail(GRPO_ERR_INVALID_ARG, "shard %d is NULL", i);
    total += shards[i]->bytes;
  }
  int dev = 0;
  if (current_device(&dev)) return grpo_internal_fail(GRPO_ERR_CUDA, "cudaGetDevice failed");
  CUdeviceptr base = 0;
  VMM_OK(vmm().Reserve(&base, total, 0, 0, 0));
  size_t off = 0;
  for (int i = 0; i < n; ++i) {
    const CUresult r = vmm().Map(base + off, shards[i]->bytes, 0, shards[i]->handle, 0);
    if (r != CUDA_SUCCESS) {
      if (off) vmm().Unmap(base, off);
      vmm().AddressFree(base, total);
      return grpo_internal_fail(GRPO_ERR_CUDA, "cuMemMap of shard %d failed with CUresult %d", i, (int)r);
    }
    off += shards[i]->bytes;
  }
  CUmemAccessDesc acc = {};
  acc.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
  acc.location.id = dev;
  acc.flags = CU_MEM_ACCESS_FLAGS_PROT_READWRITE;
  const CUresult r = vmm().SetAccess(base, total, &acc, 1);
  if (r != CUDA_SUCCESS) {
    vmm().Unmap(base, total);
    vmm().AddressFree(base, total);
    return grpo_internal_fail(GRPO_ERR_CUDA, "cuMemSetAccess failed with CUresult %d (peer access between the GPUs?)", (int)r);
  }
  {
    std::lock_guard<std::mutex> lk(g_mu);
    g_ranges[reinterpret_cast<void*>(base)] = total;
  }
  *dev_ptr_out = reinterpret_cast<void*>(base);
  return GRPO_OK;
}

extern "C" int32_t grpo_stitch_unmap(grpo_ctx* ctx, void* dev_ptr) {
  if (!ctx || !dev_ptr) return grpo_internal_fail(GRPO_ERR_INVALID_ARG, "ctx / dev_ptr is NULL");
  size_t total = 0;
  {
    std::lock_guard<std::mutex> lk(g_mu);
    auto it = g_ranges.find(dev_ptr);
    if (it == g_ranges.end()) return grpo_internal_fail(GRPO_ERR_INVALID_ARG, "pointer was not returned by grpo_stitch_map");
    total = it->second;
    g_ranges.erase(it);
  }
  if (cudaDeviceSynchronize() != cudaSuccess) return grpo_internal_fail(GRPO_ERR_CUDA, "cudaDeviceSynchronize failed");
  VMM_OK(vmm().Unmap(reinterpret_cast<CUdeviceptr>(dev_ptr), total));
  VMM_OK(vmm().AddressFree(reinterpret_cast<CUdeviceptr>(dev_ptr), total));
  return GRPO_OK;
}
