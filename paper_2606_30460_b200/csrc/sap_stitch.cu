// Stitched allocation (data plane): ONE virtual address range whose chunk c is physical memory of
// the device that owns sequence chunk c, mapped with read/write access for every device of the group.
//
// The paper moves K/V (and dK/dV, dQ) shards between ranks with grouped ncclSend/ncclRecv.
// Inside an NVLink / NVSwitch domain the B200-native form is to leave every shard where it is and let the kernels read
// it there: with q / k / v / out / dout / dq / dk / dv laid out in such ranges the attention kernels keep global token
// indices, a rank's launch (sap_attn_fwd_chunks, sap_attn_bwd_chunks) streams the K/V tiles its plan names straight
// from their owners by TMA and adds its dQ contributions into the owner's accumulator with red.global - transfer and
// compute are one kernel, and chunk pairs the plan skips are never touched.
//
// CUDA virtual-memory API (cuMemAddressReserve / cuMemCreate / cuMemMap / cuMemSetAccess), reached through
// cudaGetDriverEntryPoint like cuTensorMapEncodeTiled, so the library still links against the runtime only.
// Two forms: one process driving several devices (sap_stitched_alloc; peers must be P2P-capable, cuMemSetAccess fails
// otherwise) and one process per GPU (sap_stitched_create_local / _export_fd / _import_fd: each process creates the chunks
// it owns as exportable allocations and maps the others' through POSIX file descriptors).
#include <cstring>
#include <new>
#include <vector>
#include "sap_host.h"

struct sap_stitched {
  CUdeviceptr base = 0;
  size_t chunk_bytes = 0, total = 0;
  int32_t n_chunks = 0;
  std::vector<CUmemGenericAllocationHandle> handles;
  std::vector<int32_t> devices;
  int32_t mapped = 0;   // chunks mapped so far (for unwinding)
  // one-process-per-GPU form: chunk c is created here (owned), imported from its owner's file descriptor, or not yet mapped
  bool shared = false;
  int32_t device = -1;
  std::vector<uint8_t> state;                              // 0 unmapped, 1 owned, 2 imported
  std::vector<CUmemGenericAllocationHandle> chunk_handle;  // valid where state != 0
};

namespace sap {
namespace {

struct VmmApi {
  CUresult (*getGranularity)(size_t*, const CUmemAllocationProp*, CUmemAllocationGranularity_flags) = nullptr;
  CUresult (*addressReserve)(CUdeviceptr*, size_t, size_t, CUdeviceptr, unsigned long long) = nullptr;
  CUresult (*addressFree)(CUdeviceptr, size_t) = nullptr;
  CUresult (*create)(CUmemGenericAllocationHandle*, size_t, const CUmemAllocationProp*, unsigned long long) = nullptr;
  CUresult (*release)(CUmemGenericAllocationHandle) = nullptr;
  CUresult (*map)(CUdeviceptr, size_t, size_t, CUmemGenericAllocationHandle, unsigned long long) = nullptr;
  CUresult (*unmap)(CUdeviceptr, size_t) = nullptr;
  CUresult (*setAccess)(CUdeviceptr, size_t, const CUmemAccessDesc*, size_t) = nullptr;
  CUresult (*exportHandle)(void*, CUmemGenericAllocationHandle, CUmemAllocationHandleType, unsigned long long) = nullptr;
  CUresult (*importHandle)(CUmemGenericAllocationHandle*, void*, CUmemAllocationHandleType) = nullptr;
  bool ok = false;
};

template <class F>
bool entry(const char* name, F* fn) {
  void* p = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint(name, &p, cudaEnableDefault, &q) != cudaSuccess || !p) return false;
  *fn = reinterpret_cast<F>(p);
  return true;
}

const VmmApi& vmm() {
  static VmmApi api = [] {   // function-local static: initialised once, thread-safe
    VmmApi a;
    a.ok = entry("cuMemGetAllocationGranularity", &a.getGranularity) && entry("cuMemAddressReserve", &a.addressReserve) &&
           entry("cuMemAddressFree", &a.addressFree) && entry("cuMemCreate", &a.create) && entry("cuMemRelease", &a.release) &&
           entry("cuMemMap", &a.map) && entry("cuMemUnmap", &a.unmap) && entry("cuMemSetAccess", &a.setAccess) &&
           entry("cuMemExportToShareableHandle", &a.exportHandle) && entry("cuMemImportFromShareableHandle", &a.importHandle);
    return a;
  }();
  return api;
}

CUmemAllocationProp prop_for(int device) {
  CUmemAllocationProp p;
  std::memset(&p, 0, sizeof(p));
  p.type = CU_MEM_ALLOCATION_TYPE_PINNED;
  p.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
  p.location.id = device;
  return p;
}

int fail(CUresult r) {
  g_last_cuda_error = static_cast<int>(r);
  return SAP_ERR_CUDA;
}

}  // namespace
}  // namespace sap

using namespace sap;

extern "C" {

int sap_stitched_granularity(int device, size_t* bytes) {
  if (!bytes || device < 0) return SAP_ERR_INVALID_ARG;
  if (cudaFree(nullptr) != cudaSuccess) return SAP_ERR_NO_DEVICE;   // make sure a context exists
  const VmmApi& a = vmm();
  if (!a.ok) return SAP_ERR_UNSUPPORTED;
  const CUmemAllocationProp p = prop_for(device);
  const CUresult r = a.getGranularity(bytes, &p, CU_MEM_ALLOC_GRANULARITY_MINIMUM);
  return r == CUDA_SUCCESS ? SAP_OK : fail(r);
}

void sap_stitched_free(sap_stitched_t* s) {
  if (!s) return;
  const VmmApi& a = vmm();
  if (a.ok && s->base && s->shared) {
    for (int32_t c = 0; c < s->n_chunks; ++c)
      if (s->state[c]) {
        a.unmap(s->base + static_cast<size_t>(c) * s->chunk_bytes, s->chunk_bytes);
        a.release(s->chunk_handle[c]);   // an imported handle is a reference: the memory goes when its owner releases too
      }
    a.addressFree(s->base, s->total);
  } else if (a.ok && s->base) {
    for (int32_t c = 0; c < s->mapped; ++c) a.unmap(s->base + static_cast<size_t>(c) * s->chunk_bytes, s->chunk_bytes);
    for (CUmemGenericAllocationHandle h : s->handles) a.release(h);   // physical memory goes once it is unmapped everywhere
    a.addressFree(s->base, s->total);
  }
  delete s;
}

int sap_stitched_alloc(int32_t n_chunks, size_t chunk_bytes, const int32_t* device_of_chunk, int32_t n_access,
                       const int32_t* access_devices, sap_stitched_t** out) {
  if (!out || !device_of_chunk || !access_devices || n_chunks < 1 || n_access < 1 || chunk_bytes == 0) return SAP_ERR_INVALID_ARG;
  *out = nullptr;
  if (cudaFree(nullptr) != cudaSuccess) return SAP_ERR_NO_DEVICE;
  const VmmApi& a = vmm();
  if (!a.ok) return SAP_ERR_UNSUPPORTED;
  // a chunk boundary must be a boundary of physical allocations: chunk_bytes a multiple of every owner's granularity
  size_t gran = 1;
  for (int32_t c = 0; c < n_chunks; ++c) {
    if (device_of_chunk[c] < 0) return SAP_ERR_INVALID_ARG;
    size_t g = 0;
    int rc = sap_stitched_granularity(device_of_chunk[c], &g);
    if (rc != SAP_OK) return rc;
    if (chunk_bytes % g != 0) return SAP_ERR_UNSUPPORTED;
    if (g > gran) gran = g;
  }
  sap_stitched* s = new (std::nothrow) sap_stitched();
  if (!s) return SAP_ERR_INVALID_ARG;
  s->chunk_bytes = chunk_bytes; s->n_chunks = n_chunks; s->total = chunk_bytes * static_cast<size_t>(n_chunks);
  s->devices.assign(device_of_chunk, device_of_chunk + n_chunks);
  CUresult r = a.addressReserve(&s->base, s->total, gran, 0, 0);
  if (r != CUDA_SUCCESS) { s->base = 0; sap_stitched_free(s); return fail(r); }
  for (int32_t c = 0; c < n_chunks; ++c) {
    const CUmemAllocationProp p = prop_for(device_of_chunk[c]);
    CUmemGenericAllocationHandle h;
    if ((r = a.create(&h, chunk_bytes, &p, 0)) != CUDA_SUCCESS) { sap_stitched_free(s); return fail(r); }
    s->handles.push_back(h);
    if ((r = a.map(s->base + static_cast<size_t>(c) * chunk_bytes, chunk_bytes, 0, h, 0)) != CUDA_SUCCESS) { sap_stitched_free(s); return fail(r); }
    s->mapped = c + 1;
  }
  std::vector<CUmemAccessDesc> acc(n_access);
  for (int32_t i = 0; i < n_access; ++i) {
    std::memset(&acc[i], 0, sizeof(CUmemAccessDesc));
    acc[i].location.type = CU_MEM_LOCATION_TYPE_DEVICE;
    acc[i].location.id = access_devices[i];
    acc[i].flags = CU_MEM_ACCESS_FLAGS_PROT_READWRITE;
  }
  if ((r = a.setAccess(s->base, s->total, acc.data(), acc.size())) != CUDA_SUCCESS) { sap_stitched_free(s); return fail(r); }
  *out = s;
  return SAP_OK;
}

// ---- one process per GPU: every process reserves the whole range, creates the chunks it owns (exportable), hands their
// file descriptors to the others (SCM_RIGHTS over a Unix socket: ranks.exchange_fds) and maps theirs.
static int map_chunk(sap_stitched* s, int32_t c, CUmemGenericAllocationHandle h, uint8_t state) {
  const VmmApi& a = vmm();
  const CUdeviceptr at = s->base + static_cast<size_t>(c) * s->chunk_bytes;
  CUresult r = a.map(at, s->chunk_bytes, 0, h, 0);
  if (r != CUDA_SUCCESS) { a.release(h); return fail(r); }
  CUmemAccessDesc acc;
  std::memset(&acc, 0, sizeof(acc));
  acc.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
  acc.location.id = s->device;
  acc.flags = CU_MEM_ACCESS_FLAGS_PROT_READWRITE;
  if ((r = a.setAccess(at, s->chunk_bytes, &acc, 1)) != CUDA_SUCCESS) { a.unmap(at, s->chunk_bytes); a.release(h); return fail(r); }
  s->chunk_handle[c] = h;
  s->state[c] = state;
  return SAP_OK;
}

int sap_stitched_create_local(int32_t n_chunks, size_t chunk_bytes, int device, const uint8_t* own, sap_stitched_t** out) {
  if (!out || !own || n_chunks < 1 || chunk_bytes == 0 || device < 0) return SAP_ERR_INVALID_ARG;
  *out = nullptr;
  size_t g = 0;
  int rc = sap_stitched_granularity(device, &g);
  if (rc != SAP_OK) return rc;
  if (chunk_bytes % g != 0) return SAP_ERR_UNSUPPORTED;
  const VmmApi& a = vmm();
  sap_stitched* s = new (std::nothrow) sap_stitched();
  if (!s) return SAP_ERR_INVALID_ARG;
  s->shared = true; s->device = device;
  s->chunk_bytes = chunk_bytes; s->n_chunks = n_chunks; s->total = chunk_bytes * static_cast<size_t>(n_chunks);
  s->devices.assign(n_chunks, -1);
  s->state.assign(n_chunks, 0);
  s->chunk_handle.assign(n_chunks, 0);
  CUresult r = a.addressReserve(&s->base, s->total, g, 0, 0);
  if (r != CUDA_SUCCESS) { s->base = 0; sap_stitched_free(s); return fail(r); }
  for (int32_t c = 0; c < n_chunks; ++c) {
    if (!own[c]) continue;
    CUmemAllocationProp p = prop_for(device);
    p.requestedHandleTypes = CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR;
    CUmemGenericAllocationHandle h;
    if ((r = a.create(&h, chunk_bytes, &p, 0)) != CUDA_SUCCESS) { sap_stitched_free(s); return fail(r); }
    if ((rc = map_chunk(s, c, h, 1)) != SAP_OK) { sap_stitched_free(s); return rc; }
    s->devices[c] = device;
  }
  *out = s;
  return SAP_OK;
}

int sap_stitched_export_fd(const sap_stitched_t* s, int32_t chunk, int* fd) {
  if (!s || !fd || !s->shared || chunk < 0 || chunk >= s->n_chunks || s->state[chunk] != 1) return SAP_ERR_INVALID_ARG;
  const CUresult r = vmm().exportHandle(fd, s->chunk_handle[chunk], CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR, 0);
  return r == CUDA_SUCCESS ? SAP_OK : fail(r);
}

int sap_stitched_import_fd(sap_stitched_t* s, int32_t chunk, int fd) {
  if (!s || !s->shared || chunk < 0 || chunk >= s->n_chunks || s->state[chunk] != 0 || fd < 0) return SAP_ERR_INVALID_ARG;
  CUmemGenericAllocationHandle h;
  const CUresult r = vmm().importHandle(&h, reinterpret_cast<void*>(static_cast<uintptr_t>(fd)), CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR);
  if (r != CUDA_SUCCESS) return fail(r);
  return map_chunk(s, chunk, h, 2);
}

void* sap_stitched_ptr(const sap_stitched_t* s) { return s ? reinterpret_cast<void*>(s->base) : nullptr; }
size_t sap_stitched_bytes(const sap_stitched_t* s) { return s ? s->total : 0; }
int32_t sap_stitched_owner(const sap_stitched_t* s, int32_t chunk) {
  return (s && chunk >= 0 && chunk < s->n_chunks) ? s->devices[chunk] : -1;
}

}  // extern "C"
