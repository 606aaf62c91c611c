// C-ABI entry points that touch the GPU (include/sap.h): plan upload, forward, partial forward, LSE merge, backward,
// per-rank and per-item launches.  Argument checking + tensor-map encoding + launches only.
#include <cstdio>
#include <cstring>
#include <list>
#include <set>
#include "sap_host.h"
#include "sap_fwd.cuh"
#include "sap_fwd_pair.cuh"
#include "sap_bwd.cuh"
#include "sap_bwd_fused.cuh"
#include "sap_bwd_pair.cuh"
#include "sap_merge.cuh"

namespace sap {

// sap_debug_set_bwd_stages bits: 1 D pre-pass | 2 split dK/dV kernel | 4 split dQ kernel | 8 fused main kernel
// (+ zeroing of its fp32 dQ accumulator) | 16 dQ post pass.  Default: pre + fused + post.
constexpr int kBwdDefaultStages = 1 | 8 | 16;
constexpr size_t kMaxRangePrograms = 64;   // cached range-restricted programs per plan and kind (least recently used goes)
static inline size_t align256(size_t x) { return (x + 255) & ~size_t(255); }

thread_local int g_last_cuda_error = 0;
std::atomic<int64_t> g_launch_count{0};
std::atomic<int> g_bwd_stages{kBwdDefaultStages};
std::atomic<int> g_fwd_form{0};  // 0: pair kernel when Hq/Hkv is even, 1: always the one-head kernel (diagnostic)
std::atomic<int> g_bwd_form{0};  // 0: CTA-pair fused kernel for head_dim 128, 1: always the one-CTA fused kernel (diagnostic)

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = []() -> EncodeTiledFn {   // function-local static: initialised once, thread-safe
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess) return nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

int make_tile_map(CUtensorMap* map, const void* base, int64_t n_rows, int64_t row_elems, int box_rows) {
  EncodeTiledFn enc = get_encode_fn();
  if (!enc) { g_last_cuda_error = static_cast<int>(cudaErrorNotSupported); return SAP_ERR_CUDA; }
  cuuint64_t dims[2] = {static_cast<cuuint64_t>(row_elems), static_cast<cuuint64_t>(n_rows)};
  cuuint64_t strides[1] = {static_cast<cuuint64_t>(row_elems) * 2};
  cuuint32_t box[2] = {64, static_cast<cuuint32_t>(box_rows)};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { g_last_cuda_error = static_cast<int>(r); return SAP_ERR_CUDA; }
  return SAP_OK;
}

// Per-device one-time setup: architecture check and the opt-in shared-memory sizes of every kernel
// (cudaFuncSetAttribute is per device).  Guarded by a mutex; `*dev_out` = the current device.
template <int D>
static cudaError_t set_kernel_attributes() {
  cudaError_t e;
  const cudaFuncAttribute a = cudaFuncAttributeMaxDynamicSharedMemorySize;
  if ((e = cudaFuncSetAttribute(sap_fwd_kernel<D, false>, a, FwdSmem<D>::kTotal)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(sap_fwd_kernel<D, true>, a, FwdSmem<D>::kTotal)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(sap_fwd_pair_kernel<D, false>, a, FwdPairSmem<D>::kTotal)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(sap_fwd_pair_kernel<D, true>, a, FwdPairSmem<D>::kTotal)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(sap_bwd_dq_kernel<D>, a, DqSmem<D>::kTotal)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(sap_bwd_dkv_kernel<D>, a, DkvSmem<D>::kTotal)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(sap_bwd_fused_kernel<D>, a, FusedSmem<D>::kTotal)) != cudaSuccess) return e;
  return cudaSuccess;
}

// Per-device state of the persistent kernels: the SM count and two pools of {next, done} counter pairs (zero between
// launches: the last CTA of a launch re-arms its pair).  A pair must serve one launch at a time.
//   eager pool   : launches outside stream capture take its pairs round-robin, so two of them hold the same pair only
//                  if kSchedSlots forward launches are in flight on the device at once.
//   capture pool : a launch recorded into a CUDA graph keeps its pair for the life of the graph and runs at replay
//                  time, when the host cannot pick one.  Such launches draw from a pool of their own, so a replay
//                  never meets an eager launch on its pair; two graphs share a pair only once more than kSchedSlots
//                  forward launches have been captured in the process (round-robin again).
// The kernel traps if it finds that its pair was shared (sap_fwd_pair.cuh, last lines).
constexpr int kSchedSlots = 4096;
struct DeviceSched { int n_sms = 0; int* pool = nullptr; std::atomic<unsigned> seq{0}, seq_capture{0}; };
static DeviceSched g_sched[64];

static int* next_sched_pair(int dev, cudaStream_t stream) {
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(stream, &cs) != cudaSuccess) { cudaGetLastError(); cs = cudaStreamCaptureStatusNone; }
  DeviceSched& d = g_sched[dev];
  if (cs == cudaStreamCaptureStatusActive) return d.pool + 2 * (kSchedSlots + d.seq_capture.fetch_add(1) % kSchedSlots);
  return d.pool + 2 * (d.seq.fetch_add(1) % kSchedSlots);
}

int ensure_device(int* dev_out) {
  static std::mutex mu;
  static std::set<int> ready, wrong_arch;
  int dev = 0;
  SAP_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev_out) *dev_out = dev;
  if (dev < 0 || dev >= 64) return SAP_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(mu);
  if (ready.count(dev)) return SAP_OK;
  if (wrong_arch.count(dev)) return SAP_ERR_WRONG_ARCH;
  int major = 0;
  SAP_CUDA_CHECK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  if (major != 10) { wrong_arch.insert(dev); return SAP_ERR_WRONG_ARCH; }
  SAP_CUDA_CHECK(set_kernel_attributes<64>());
  SAP_CUDA_CHECK(set_kernel_attributes<128>());
  SAP_CUDA_CHECK(cudaFuncSetAttribute(sap_bwd_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, PairSmem::kTotal));
  SAP_CUDA_CHECK(cudaDeviceGetAttribute(&g_sched[dev].n_sms, cudaDevAttrMultiProcessorCount, dev));
  if (!g_sched[dev].pool) {
    SAP_CUDA_CHECK(cudaMalloc(&g_sched[dev].pool, 2 * 2 * kSchedSlots * sizeof(int)));   // eager pool | capture pool
    SAP_CUDA_CHECK(cudaMemset(g_sched[dev].pool, 0, 2 * 2 * kSchedSlots * sizeof(int)));
  }
  ready.insert(dev);
  return SAP_OK;
}

void free_program(DevProgram& dev) {
  if (dev.tiles) cudaFree(dev.tiles);
  if (dev.segs) cudaFree(dev.segs);
  dev = DevProgram();
}

// Synchronous upload (sap_plan_upload).  Frees what it allocated when a later step fails.
int upload_program(const TileProgram& host, DevProgram& dev) {
  dev = DevProgram();
  dev.n_tiles = static_cast<int32_t>(host.tiles.size());
  const size_t tb = host.tiles.size() * sizeof(TileDesc), sb = (host.segs.size() + 1) * sizeof(SegDesc);
  cudaError_t e = cudaMalloc(&dev.tiles, tb ? tb : sizeof(TileDesc));
  if (e == cudaSuccess) e = cudaMalloc(&dev.segs, sb);
  if (e == cudaSuccess && tb) e = cudaMemcpy(dev.tiles, host.tiles.data(), tb, cudaMemcpyHostToDevice);
  if (e == cudaSuccess && !host.segs.empty())
    e = cudaMemcpy(dev.segs, host.segs.data(), host.segs.size() * sizeof(SegDesc), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { free_program(dev); SAP_CUDA_CHECK(e); }
  return SAP_OK;
}

// Stream-ordered upload of a range-restricted program: no device synchronisation.  `host` must stay alive until the
// copies have run (it lives in the cache entry); `ready` is recorded behind the copies for uses on other streams.
static int upload_program_async(const TileProgram& host, DevProgram& dev, cudaEvent_t* ready, cudaStream_t stream) {
  dev = DevProgram();
  dev.n_tiles = static_cast<int32_t>(host.tiles.size());
  const size_t tb = host.tiles.size() * sizeof(TileDesc), sb = (host.segs.size() + 1) * sizeof(SegDesc);
  cudaError_t e = cudaMallocAsync(reinterpret_cast<void**>(&dev.tiles), tb ? tb : sizeof(TileDesc), stream);
  if (e == cudaSuccess) e = cudaMallocAsync(reinterpret_cast<void**>(&dev.segs), sb, stream);
  if (e == cudaSuccess && tb) e = cudaMemcpyAsync(dev.tiles, host.tiles.data(), tb, cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess && !host.segs.empty())
    e = cudaMemcpyAsync(dev.segs, host.segs.data(), host.segs.size() * sizeof(SegDesc), cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(ready, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventRecord(*ready, stream);
  if (e != cudaSuccess) {
    if (dev.tiles) cudaFreeAsync(dev.tiles, stream);
    if (dev.segs) cudaFreeAsync(dev.segs, stream);
    dev = DevProgram();
    SAP_CUDA_CHECK(e);
  }
  return SAP_OK;
}

static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// Common checks of the attention calls: dims, the caller's length against the plan's (a plan built for another length
// would make the kernels read out of bounds), device setup, and that the plan's device mirror lives on this device.
static int check_call(sap_plan_t* plan, int64_t n_tokens, int Hq, int Hkv, int d, float scale, bool need_upload = true) {
  if (!plan) return SAP_ERR_INVALID_ARG;
  if (Hq < 1 || Hkv < 1 || !(scale > 0.f)) return SAP_ERR_INVALID_ARG;
  if ((d != 64 && d != 128) || Hq % Hkv != 0) return SAP_ERR_UNSUPPORTED;
  if (n_tokens != plan->n_tokens) return SAP_ERR_PLAN_MISMATCH;
  int dev = 0, rc;
  if ((rc = ensure_device(&dev)) != SAP_OK) return rc;
  if (need_upload && (rc = sap_plan_upload(plan)) != SAP_OK) return rc;
  const PlanDevice* pd = static_cast<const PlanDevice*>(plan->dev_state);
  if (pd && pd->uploaded && pd->device != dev) return SAP_ERR_PLAN_MISMATCH;
  return SAP_OK;
}

// Row pairs pay once there are many work items per SM (measured on the Table 2 shape, 16 heads MHA: 128K tokens 12.27 -> 11.50
// ms; 32K 0.69 -> 0.70 ms; 8K 0.110 -> 0.117 ms - there the one-head kernel's two smaller CTAs per SM spread the work better).
static bool use_row_pairs(int n_tiles2, int Hq) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || n_tiles2 <= 0) return false;
  return static_cast<int64_t>(n_tiles2) * Hq >= 16ll * g_sched[dev].n_sms;
}

// `prog2` (optional): the same work as `prog` in 256-row Q tiles, for the row-pair form of the pair kernel.
template <int D, bool PARTIAL>
static int launch_fwd(const DevProgram& prog, const void* q, const void* k, const void* v, const int32_t* cu,
                      const sap_plan_t* plan, void* out, float* out_f32, float* lse, int Hq, int Hkv, float scale,
                      cudaStream_t stream, const DevProgram* prog2 = nullptr) {
  if (prog.n_tiles == 0) return SAP_OK;
  CUtensorMap mq, mk, mv;
  int rc;
  if ((rc = make_tile_map(&mq, q, plan->n_tokens, (int64_t)Hq * D)) != SAP_OK) return rc;
  if ((rc = make_tile_map(&mk, k, plan->n_tokens, (int64_t)Hkv * D)) != SAP_OK) return rc;
  if ((rc = make_tile_map(&mv, v, plan->n_tokens, (int64_t)Hkv * D)) != SAP_OK) return rc;
  if ((Hq / Hkv) % 2 == 0 && g_fwd_form.load() == 0) {  // two q-heads of a GQA group per CTA share the K/V stream
    // persistent: one CTA per SM, work items handed out in launch order (kv-head-major, longest tile first)
    int dev = 0;
    SAP_CUDA_CHECK(cudaGetDevice(&dev));
    const int n_work = prog.n_tiles * (Hq / 2);
    const unsigned grid = static_cast<unsigned>(n_work < g_sched[dev].n_sms ? n_work : g_sched[dev].n_sms);
    sap_fwd_pair_kernel<D, PARTIAL><<<grid, kFwdPairThreads, FwdPairSmem<D>::kTotal, stream>>>(
        mq, mk, mv, prog.tiles, prog.segs, cu, plan->n_docs, static_cast<__nv_bfloat16*>(out), out_f32, lse,
        plan->n_tokens, Hq, Hkv, scale * kLog2e, prog.n_tiles, n_work, next_sched_pair(dev, stream), 0);
  } else if (prog2 && prog2->n_tiles > 0 && ((g_fwd_form.load() == 0 && use_row_pairs(prog2->n_tiles, Hq)) || g_fwd_form.load() == 2)) {
    // odd Hq/Hkv (MHA): the same persistent kernel, its two units = the two 128-row halves of a 256-row tile of ONE q-head
    int dev = 0;
    SAP_CUDA_CHECK(cudaGetDevice(&dev));
    const int n_work = prog2->n_tiles * Hq;
    const unsigned grid = static_cast<unsigned>(n_work < g_sched[dev].n_sms ? n_work : g_sched[dev].n_sms);
    sap_fwd_pair_kernel<D, PARTIAL><<<grid, kFwdPairThreads, FwdPairSmem<D>::kTotal, stream>>>(
        mq, mk, mv, prog2->tiles, prog2->segs, cu, plan->n_docs, static_cast<__nv_bfloat16*>(out), out_f32, lse,
        plan->n_tokens, Hq, Hkv, scale * kLog2e, prog2->n_tiles, n_work, next_sched_pair(dev, stream), 1);
  } else {
    const unsigned grid = static_cast<unsigned>(prog.n_tiles) * Hq;
    sap_fwd_kernel<D, PARTIAL><<<grid, kFwdThreads, FwdSmem<D>::kTotal, stream>>>(
        mq, mk, mv, prog.tiles, prog.segs, cu, plan->n_docs, static_cast<__nv_bfloat16*>(out), out_f32, lse,
        plan->n_tokens, Hq, Hkv, scale * kLog2e);
  }
  g_launch_count.fetch_add(1);
  SAP_CUDA_CHECK(cudaGetLastError());
  return SAP_OK;
}

// a6: the fused main kernel over a KV-stationary program.  head_dim 128 runs on CTA pairs over a 256-key program
// `prog2`, head_dim 64 (and the diagnostic form) on single CTAs over a 128-key program `prog1`.
static inline bool use_pair_kernel(int d) { return d == 128 && g_bwd_form.load() == 0; }

template <int D>
static int launch_bwd_main(const DevProgram& prog1, const DevProgram& prog2, const void* dout, const void* q, const void* k,
                           const void* v, const float* lse, const int32_t* cu, const sap_plan_t* plan, void* dk, void* dv,
                           int Hq, int Hkv, float scale, const float* dsum, float* dq_acc, cudaStream_t stream) {
  const int64_t N = plan->n_tokens;
  CUtensorMap mq64, mdo64, mk128, mv128;
  int rc;
  if ((rc = make_tile_map(&mq64, q, N, (int64_t)Hq * D, kBwdN)) != SAP_OK) return rc;
  if ((rc = make_tile_map(&mdo64, dout, N, (int64_t)Hq * D, kBwdN)) != SAP_OK) return rc;
  if ((rc = make_tile_map(&mk128, k, N, (int64_t)Hkv * D, kTile)) != SAP_OK) return rc;
  if ((rc = make_tile_map(&mv128, v, N, (int64_t)Hkv * D, kTile)) != SAP_OK) return rc;
  if (use_pair_kernel(D)) {
    if (prog2.n_tiles == 0) return SAP_OK;
    CUtensorMap mq32, mdo32;
    if ((rc = make_tile_map(&mq32, q, N, (int64_t)Hq * D, 32)) != SAP_OK) return rc;
    if ((rc = make_tile_map(&mdo32, dout, N, (int64_t)Hq * D, 32)) != SAP_OK) return rc;
    sap_bwd_pair_kernel<<<2u * static_cast<unsigned>(prog2.n_tiles) * Hkv, kPairThreads, PairSmem::kTotal, stream>>>(
        mq32, mdo32, mq64, mdo64, mk128, mv128, prog2.tiles, prog2.segs, cu, plan->n_docs, lse, dsum, dq_acc,
        static_cast<__nv_bfloat16*>(dk), static_cast<__nv_bfloat16*>(dv), plan->n_tokens, Hq, Hkv, scale, scale * kLog2e);
  } else {
    if (prog1.n_tiles == 0) return SAP_OK;
    sap_bwd_fused_kernel<D><<<static_cast<unsigned>(prog1.n_tiles) * Hkv, kFusedThreads, FusedSmem<D>::kTotal, stream>>>(
        mq64, mdo64, mk128, mv128, prog1.tiles, prog1.segs, cu, plan->n_docs, lse, dsum, dq_acc,
        static_cast<__nv_bfloat16*>(dk), static_cast<__nv_bfloat16*>(dv), plan->n_tokens, Hq, Hkv, scale, scale * kLog2e);
  }
  g_launch_count.fetch_add(1);
  SAP_CUDA_CHECK(cudaGetLastError());
  return SAP_OK;
}

// a5 for tokens [t0, t0 + nt): D = rowsum(dO * O); optionally zero the dQ accumulator rows
template <int D>
static int launch_bwd_pre(const void* dout, const void* out, int64_t N, int Hq, int64_t t0, int64_t nt, float* dsum,
                          float* dq_acc, bool zero_acc, cudaStream_t stream) {
  if (nt == 0) return SAP_OK;
  const int64_t want = (nt * Hq * (D / 8) + kPreThreads - 1) / kPreThreads;
  const unsigned grid = static_cast<unsigned>(want < 148 * 16 ? want : 148 * 16);
  sap_bwd_pre_kernel<D><<<grid, kPreThreads, 0, stream>>>(static_cast<const __nv_bfloat16*>(dout),
                                                          static_cast<const __nv_bfloat16*>(out), dsum, N, Hq, t0, nt);
  g_launch_count.fetch_add(1);
  SAP_CUDA_CHECK(cudaGetLastError());
  if (zero_acc) SAP_CUDA_CHECK(cudaMemsetAsync(dq_acc + t0 * Hq * D, 0, static_cast<size_t>(nt) * Hq * D * sizeof(float), stream));
  return SAP_OK;
}

// a7 for tokens [t0, t0 + nt): dq = bf16(scale * dq_acc)
static int launch_bwd_post(const float* dq_acc, void* dq, int Hq, int d, int64_t t0, int64_t nt, float scale, cudaStream_t stream) {
  const int64_t n8 = nt * Hq * d / 8;
  if (n8 == 0) return SAP_OK;
  const int64_t want = (n8 + kPostThreads - 1) / kPostThreads;
  const unsigned grid = static_cast<unsigned>(want < 148 * 16 ? want : 148 * 16);
  sap_bwd_post_kernel<<<grid, kPostThreads, 0, stream>>>(dq_acc + t0 * Hq * d,
                                                         static_cast<__nv_bfloat16*>(dq) + t0 * Hq * d, n8, scale);
  g_launch_count.fetch_add(1);
  SAP_CUDA_CHECK(cudaGetLastError());
  return SAP_OK;
}

template <int D>
static int launch_bwd(const PlanDevice* pd, const void* dout, const void* q, const void* k, const void* v,
                      const void* out, const float* lse, const int32_t* cu, const sap_plan_t* plan, void* dq, void* dk,
                      void* dv, int Hq, int Hkv, float scale, float* dsum, float* dq_acc, cudaStream_t stream) {
  const int64_t N = plan->n_tokens;
  int rc;
  const int stages = g_bwd_stages.load();
  if (stages & 1)
    if ((rc = launch_bwd_pre<D>(dout, out, N, Hq, 0, N, dsum, dq_acc, false, stream)) != SAP_OK) return rc;
  if (stages & 8) {  // a6 fused: dK, dV and the fp32 dQ accumulator in one pass (5 GEMMs per tile pair)
    SAP_CUDA_CHECK(cudaMemsetAsync(dq_acc, 0, static_cast<size_t>(N) * Hq * D * sizeof(float), stream));
    if ((rc = launch_bwd_main<D>(pd->kv, pd->kv2, dout, q, k, v, lse, cu, plan, dk, dv, Hq, Hkv, scale, dsum, dq_acc, stream)) != SAP_OK) return rc;
  }
  if (stages & 16)
    if ((rc = launch_bwd_post(dq_acc, dq, Hq, D, 0, N, scale, stream)) != SAP_OK) return rc;
  if (stages & 6) {  // the split, atomics-free form (diagnostic): 7 GEMMs per tile pair
    CUtensorMap mq128, mdo128, mk64, mv64, mq64, mdo64, mk128, mv128;
    if ((rc = make_tile_map(&mq128, q, N, (int64_t)Hq * D, kTile)) != SAP_OK) return rc;
    if ((rc = make_tile_map(&mdo128, dout, N, (int64_t)Hq * D, kTile)) != SAP_OK) return rc;
    if ((rc = make_tile_map(&mk64, k, N, (int64_t)Hkv * D, kBwdN)) != SAP_OK) return rc;
    if ((rc = make_tile_map(&mv64, v, N, (int64_t)Hkv * D, kBwdN)) != SAP_OK) return rc;
    if ((rc = make_tile_map(&mq64, q, N, (int64_t)Hq * D, kBwdN)) != SAP_OK) return rc;
    if ((rc = make_tile_map(&mdo64, dout, N, (int64_t)Hq * D, kBwdN)) != SAP_OK) return rc;
    if ((rc = make_tile_map(&mk128, k, N, (int64_t)Hkv * D, kTile)) != SAP_OK) return rc;
    if ((rc = make_tile_map(&mv128, v, N, (int64_t)Hkv * D, kTile)) != SAP_OK) return rc;
    if (stages & 2) {
      sap_bwd_dkv_kernel<D><<<static_cast<unsigned>(pd->kv.n_tiles) * Hkv, kDkvThreads, DkvSmem<D>::kTotal, stream>>>(
          mq64, mdo64, mk128, mv128, pd->kv.tiles, pd->kv.segs, cu, plan->n_docs, lse, dsum,
          static_cast<__nv_bfloat16*>(dk), static_cast<__nv_bfloat16*>(dv), plan->n_tokens, Hq, Hkv, scale, scale * kLog2e);
      g_launch_count.fetch_add(1);
      SAP_CUDA_CHECK(cudaGetLastError());
    }
    if (stages & 4) {
      sap_bwd_dq_kernel<D><<<static_cast<unsigned>(pd->fwd.n_tiles) * Hq, kDqThreads, DqSmem<D>::kTotal, stream>>>(
          mq128, mdo128, mk64, mv64, pd->fwd.tiles, pd->fwd.segs, cu, plan->n_docs, lse, dsum,
          static_cast<__nv_bfloat16*>(dq), plan->n_tokens, Hq, Hkv, scale, scale * kLog2e);
      g_launch_count.fetch_add(1);
      SAP_CUDA_CHECK(cudaGetLastError());
    }
  }
  return SAP_OK;
}

// Range-restricted programs, built on first use of a range and kept with the plan (at most kMaxRangePrograms per
// kind; the least recently used one that no call and no CUDA graph holds is evicted).  Uploads and evictions are
// ordered on streams: no synchronisation.
static void destroy_range_program(RangeProgram& e) {   // immediate: the caller knows that nothing uses it any more
  free_program(e.dev);
  if (e.ready) cudaEventDestroy(e.ready);
  for (auto& u : e.used) cudaEventDestroy(u.second);
  e.used.clear();
}

// Frees an evicted program on `stream`, behind the last kernels that read it on every stream that used it.
static void retire_range_program(RangeProgram& e, cudaStream_t stream) {
  for (auto& u : e.used)
    if (u.first != stream) cudaStreamWaitEvent(stream, u.second, 0);
  if (e.stream != stream && e.ready) cudaStreamWaitEvent(stream, e.ready, 0);
  if (e.dev.tiles) cudaFreeAsync(e.dev.tiles, stream);
  if (e.dev.segs) cudaFreeAsync(e.dev.segs, stream);
  e.dev = DevProgram();
  destroy_range_program(e);   // cudaEventDestroy of a pending event is legal: the waits above are already enqueued
}

static bool stream_is_capturing(cudaStream_t stream) {
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(stream, &cs) != cudaSuccess) { cudaGetLastError(); return false; }
  return cs == cudaStreamCaptureStatusActive;
}

// One call's hold on a cached range program: acquire() looks it up (or builds and uploads it) and pins it, the
// destructor - after the call has enqueued its kernels - records the event eviction waits for and lets go.
struct RangeUse {
  sap_plan_t* plan = nullptr;
  RangeProgram* entry = nullptr;
  cudaStream_t stream = nullptr;
  bool capturing = false;
  DevProgram prog;

  int acquire(sap_plan_t* p, int kind, int32_t a, int32_t b, cudaStream_t st) {
    plan = p; stream = st;
    capturing = stream_is_capturing(st);
    PlanDevice* pd = static_cast<PlanDevice*>(plan->dev_state);
    std::lock_guard<std::mutex> lock(plan->mu);
    auto& cache = pd->ranges[kind];
    const auto key = std::make_pair(a, b);
    RangeProgram* hit = nullptr;
    for (auto it = cache.begin(); it != cache.end(); ++it)
      if (it->key == key) { cache.splice(cache.begin(), cache, it); hit = &cache.front(); break; }
    if (!hit) {
      // building a program allocates (cudaMallocAsync) and copies from pageable host memory: neither belongs in a graph
      if (capturing) return SAP_ERR_UNSUPPORTED;
      if (cache.size() >= kMaxRangePrograms)
        for (auto it = cache.end(); it != cache.begin();) {   // least recently used first; held entries stay
          --it;
          if (it->pins == 0 && !it->held_by_graph) { retire_range_program(*it, stream); cache.erase(it); break; }
        }
      cache.emplace_front();
      RangeProgram& e = cache.front();
      e.key = key;
      const int32_t kv_rows = (kind == kRangeKvPair || kind == kRangeItemsKvPair) ? 2 * kTile : kTile;
      switch (kind) {
        case kRangeItemsQ: build_q_program(*plan, a, b, e.host); break;                                               // partial forward, every row
        case kRangeItemsQDrop: build_q_program(*plan, a, b, e.host, true); break;                                     // ... touched Q tiles only
        case kRangeQ: build_q_program(*plan, plan->chunk_offsets[a], plan->chunk_offsets[b], e.host, true); break;    // q-chunks
        case kRangeQ2: build_q_program(*plan, plan->chunk_offsets[a], plan->chunk_offsets[b], e.host, true, 2 * kTile); break;   // ... in 256-row tiles
        case kRangeKv: case kRangeKvPair: build_kv_program(*plan, e.host, a, b, kv_rows); break;                      // kv-chunks
        default: build_kv_program(*plan, e.host, 0, -1, kv_rows, a, b, true); break;                                  // items, KV-stationary
      }
      e.stream = stream;
      int rc = upload_program_async(e.host, e.dev, &e.ready, stream);
      if (rc != SAP_OK) { cache.pop_front(); return rc; }
      hit = &e;
    }
    if (hit->stream != stream)   // a capturing stream may wait for an event from outside its graph only as an external one
      SAP_CUDA_CHECK(cudaStreamWaitEvent(stream, hit->ready, capturing ? cudaEventWaitExternal : 0));
    if (capturing) hit->held_by_graph = true;   // the graph will read it at every replay: never evicted
    ++hit->pins;
    entry = hit;
    prog = hit->dev;
    return SAP_OK;
  }

  ~RangeUse() {
    if (!entry) return;
    std::lock_guard<std::mutex> lock(plan->mu);
    --entry->pins;
    if (capturing) return;   // held_by_graph keeps it; an event recorded here would belong to the graph
    cudaEvent_t ev = nullptr;
    for (auto& u : entry->used) if (u.first == stream) ev = u.second;
    if (!ev) {
      if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); entry->held_by_graph = true; return; }
      entry->used.emplace_back(stream, ev);
    }
    if (cudaEventRecord(ev, stream) != cudaSuccess) { cudaGetLastError(); entry->held_by_graph = true; }   // cannot order a free: keep it
  }
};

static inline bool chunk_range_ok(const sap_plan_t* plan, int32_t a, int32_t b) { return a >= 0 && b >= a && b <= plan->n_chunks; }
static inline bool item_range_ok(const sap_plan_t* plan, int32_t a, int32_t b) { return a >= 0 && b >= a && b <= (int32_t)plan->items.size(); }

static int bwd_ws(const sap_plan_t* plan, int Hq, int Hkv, int d, void* workspace, size_t bytes, float** dsum, float** dq_acc) {
  if (!aligned16(workspace)) return SAP_ERR_UNSUPPORTED;
  if (!workspace || bytes < sap_workspace_bytes(plan, Hq, Hkv, d, SAP_PASS_BWD)) return SAP_ERR_WORKSPACE_TOO_SMALL;
  *dsum = static_cast<float*>(workspace);
  *dq_acc = reinterpret_cast<float*>(static_cast<uint8_t*>(workspace) + align256(static_cast<size_t>(plan->n_tokens) * Hq * sizeof(float)));
  return SAP_OK;
}

// dst (+)= alpha * src, elementwise, fp32 or bf16 on either side; 8 elements per thread and step
template <bool DST_BF16, bool SRC_BF16>
__global__ void __launch_bounds__(256)
sap_axpy_kernel(void* dst, const void* src, int64_t n8, float alpha, int accumulate) {
  const int64_t stride = static_cast<int64_t>(gridDim.x) * blockDim.x;
  for (int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; i < n8; i += stride) {
    float s[8], d[8];
    if (SRC_BF16) {
      const uint4 w = reinterpret_cast<const uint4*>(src)[i];
      const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
      for (int e = 0; e < 4; ++e) { s[2 * e] = __uint_as_float(ww[e] << 16); s[2 * e + 1] = __uint_as_float(ww[e] & 0xffff0000u); }
    } else {
      const float4 a = reinterpret_cast<const float4*>(src)[2 * i], b = reinterpret_cast<const float4*>(src)[2 * i + 1];
      s[0] = a.x; s[1] = a.y; s[2] = a.z; s[3] = a.w; s[4] = b.x; s[5] = b.y; s[6] = b.z; s[7] = b.w;
    }
#pragma unroll
    for (int e = 0; e < 8; ++e) d[e] = 0.f;
    if (accumulate) {
      if (DST_BF16) {
        const uint4 w = reinterpret_cast<const uint4*>(dst)[i];
        const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
        for (int e = 0; e < 4; ++e) { d[2 * e] = __uint_as_float(ww[e] << 16); d[2 * e + 1] = __uint_as_float(ww[e] & 0xffff0000u); }
      } else {
        const float4 a = reinterpret_cast<const float4*>(dst)[2 * i], b = reinterpret_cast<const float4*>(dst)[2 * i + 1];
        d[0] = a.x; d[1] = a.y; d[2] = a.z; d[3] = a.w; d[4] = b.x; d[5] = b.y; d[6] = b.z; d[7] = b.w;
      }
    }
#pragma unroll
    for (int e = 0; e < 8; ++e) d[e] = fmaf(alpha, s[e], d[e]);
    if (DST_BF16) {
      uint4 w;
      w.x = pack_bf16x2(d[0], d[1]); w.y = pack_bf16x2(d[2], d[3]); w.z = pack_bf16x2(d[4], d[5]); w.w = pack_bf16x2(d[6], d[7]);
      reinterpret_cast<uint4*>(dst)[i] = w;
    } else {
      reinterpret_cast<float4*>(dst)[2 * i] = make_float4(d[0], d[1], d[2], d[3]);
      reinterpret_cast<float4*>(dst)[2 * i + 1] = make_float4(d[4], d[5], d[6], d[7]);
    }
  }
}

}  // namespace sap

using namespace sap;

extern "C" {

int sap_last_cuda_error(void) { return g_last_cuda_error; }
int64_t sap_launch_count(void) { return g_launch_count.load(); }
#ifdef SAP_TRACE
int sap_debug_read_trace(unsigned long long* host_out) {
  return (int)cudaMemcpyFromSymbol(host_out, g_sap_trace, sizeof(unsigned long long) * 128 * 64);
}
int sap_debug_clear_trace(void) {   // zero everything; slots 21 / 53 (atomicMin stamps) start at the maximum
  static unsigned long long h[128 * 64];
  for (int i = 0; i < 128; ++i) for (int s2 = 0; s2 < 64; ++s2) h[i * 64 + s2] = (s2 == 21 || s2 == 53) ? ~0ull : 0ull;
  return (int)cudaMemcpyToSymbol(g_sap_trace, h, sizeof(h));
}
#endif
int sap_debug_set_fwd_form(int form) { return g_fwd_form.exchange(form == 1 || form == 2 ? form : 0); }
int sap_debug_set_bwd_form(int form) { return g_bwd_form.exchange(form ? 1 : 0); }
int sap_debug_set_bwd_stages(int mask) { return g_bwd_stages.exchange(mask < 0 ? kBwdDefaultStages : (mask & 31)); }

int sap_plan_upload(sap_plan_t* plan) {
  if (!plan) return SAP_ERR_INVALID_ARG;
  int dev = 0;
  int rc = ensure_device(&dev);
  if (rc != SAP_OK) return rc;
  std::lock_guard<std::mutex> lock(plan->mu);
  PlanDevice* pd = static_cast<PlanDevice*>(plan->dev_state);
  if (pd && pd->uploaded) return pd->device == dev ? SAP_OK : SAP_ERR_PLAN_MISMATCH;   // a plan's mirror lives on one device
  if (!pd) { pd = new PlanDevice(); plan->dev_state = pd; }
  pd->device = dev;
  if ((rc = upload_program(plan->fwd, pd->fwd)) == SAP_OK && (rc = upload_program(plan->kv, pd->kv)) == SAP_OK &&
      (rc = upload_program(plan->kv2, pd->kv2)) == SAP_OK)
    rc = upload_program(plan->fwd2, pd->fwd2);
  if (rc != SAP_OK) {  // leave nothing half-uploaded behind: a retry starts from scratch
    free_program(pd->fwd); free_program(pd->kv); free_program(pd->kv2); free_program(pd->fwd2);
    return rc;
  }
  pd->uploaded = true;
  return SAP_OK;
}

void sap_plan_destroy(sap_plan_t* plan) {
  if (!plan) return;
  PlanDevice* pd = static_cast<PlanDevice*>(plan->dev_state);
  if (pd) {
    int cur = -1;
    const bool switched = pd->uploaded && cudaGetDevice(&cur) == cudaSuccess && cur != pd->device && cudaSetDevice(pd->device) == cudaSuccess;
    free_program(pd->fwd);
    free_program(pd->kv);
    free_program(pd->kv2);
    free_program(pd->fwd2);
    for (auto& cache : pd->ranges)
      for (auto& e : cache) destroy_range_program(e);
    if (switched) cudaSetDevice(cur);
    delete pd;
  }
  delete plan;
}

size_t sap_workspace_bytes(const sap_plan_t* plan, int n_q_heads, int n_kv_heads, int head_dim, int pass) {
  (void)n_kv_heads;
  if (!plan || pass != SAP_PASS_BWD) return 0;
  // D = rowsum(dO * O), fp32 [Hq, N]  |  dQ accumulator, fp32 [N, Hq, d]
  return align256(static_cast<size_t>(plan->n_tokens) * n_q_heads * sizeof(float)) +
         static_cast<size_t>(plan->n_tokens) * n_q_heads * head_dim * sizeof(float);
}

int sap_attn_fwd(const void* q, const void* k, const void* v, const int32_t* cu_seqlens_dev, sap_plan_t* plan,
                 int64_t n_tokens, void* out, float* lse, int n_q_heads, int n_kv_heads, int head_dim, float softmax_scale,
                 void* workspace, size_t workspace_bytes, void* cuda_stream) {
  (void)workspace; (void)workspace_bytes;
  if (!q || !k || !v || !cu_seqlens_dev || !out || !lse) return SAP_ERR_INVALID_ARG;
  int rc = check_call(plan, n_tokens, n_q_heads, n_kv_heads, head_dim, softmax_scale);
  if (rc != SAP_OK) return rc;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out)) return SAP_ERR_UNSUPPORTED;
  const PlanDevice* pd = static_cast<const PlanDevice*>(plan->dev_state);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (head_dim == 128)
    return launch_fwd<128, false>(pd->fwd, q, k, v, cu_seqlens_dev, plan, out, nullptr, lse, n_q_heads, n_kv_heads, softmax_scale, st, &pd->fwd2);
  return launch_fwd<64, false>(pd->fwd, q, k, v, cu_seqlens_dev, plan, out, nullptr, lse, n_q_heads, n_kv_heads, softmax_scale, st, &pd->fwd2);
}

int sap_attn_fwd_partial(const void* q, const void* k, const void* v, const int32_t* cu_seqlens_dev, sap_plan_t* plan,
                         int64_t n_tokens, int32_t item_begin, int32_t item_end, float* out_f32, float* lse, int n_q_heads,
                         int n_kv_heads, int head_dim, float softmax_scale, void* cuda_stream) {
  if (!q || !k || !v || !cu_seqlens_dev || !out_f32 || !lse) return SAP_ERR_INVALID_ARG;
  int rc = check_call(plan, n_tokens, n_q_heads, n_kv_heads, head_dim, softmax_scale);
  if (rc != SAP_OK) return rc;
  if (!item_range_ok(plan, item_begin, item_end)) return SAP_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out_f32)) return SAP_ERR_UNSUPPORTED;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  RangeUse use;
  if ((rc = use.acquire(plan, kRangeItemsQ, item_begin, item_end, st)) != SAP_OK) return rc;
  const DevProgram& prog = use.prog;
  if (head_dim == 128)
    return launch_fwd<128, true>(prog, q, k, v, cu_seqlens_dev, plan, nullptr, out_f32, lse, n_q_heads, n_kv_heads, softmax_scale, st);
  return launch_fwd<64, true>(prog, q, k, v, cu_seqlens_dev, plan, nullptr, out_f32, lse, n_q_heads, n_kv_heads, softmax_scale, st);
}

int sap_attn_fwd_items(const void* q, const void* k, const void* v, const int32_t* cu_seqlens_dev, sap_plan_t* plan,
                       int64_t n_tokens, int32_t item_begin, int32_t item_end, float* out_f32, float* lse, int n_q_heads,
                       int n_kv_heads, int head_dim, float softmax_scale, void* cuda_stream) {
  if (!q || !k || !v || !cu_seqlens_dev || !out_f32 || !lse) return SAP_ERR_INVALID_ARG;
  int rc = check_call(plan, n_tokens, n_q_heads, n_kv_heads, head_dim, softmax_scale);
  if (rc != SAP_OK) return rc;
  if (!item_range_ok(plan, item_begin, item_end)) return SAP_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out_f32)) return SAP_ERR_UNSUPPORTED;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  RangeUse use;
  if ((rc = use.acquire(plan, kRangeItemsQDrop, item_begin, item_end, st)) != SAP_OK) return rc;
  const DevProgram& prog = use.prog;
  if (head_dim == 128)
    return launch_fwd<128, true>(prog, q, k, v, cu_seqlens_dev, plan, nullptr, out_f32, lse, n_q_heads, n_kv_heads, softmax_scale, st);
  return launch_fwd<64, true>(prog, q, k, v, cu_seqlens_dev, plan, nullptr, out_f32, lse, n_q_heads, n_kv_heads, softmax_scale, st);
}

int sap_lse_merge(const float* o_a, const float* lse_a, const float* o_b, const float* lse_b, void* o_out,
                  int out_is_bf16, float* lse_out, int64_t n_tokens, int n_q_heads, int head_dim, int64_t row_begin,
                  int64_t row_end, void* cuda_stream) {
  if (!o_a || !lse_a || !o_b || !lse_b || !o_out || !lse_out) return SAP_ERR_INVALID_ARG;
  if (n_tokens < 1 || n_q_heads < 1 || row_begin < 0 || row_end < row_begin || row_end > n_tokens) return SAP_ERR_INVALID_ARG;
  if (head_dim < 4 || head_dim % 4 != 0) return SAP_ERR_UNSUPPORTED;
  if (!aligned16(o_a) || !aligned16(o_b) || (reinterpret_cast<uintptr_t>(o_out) & 7u)) return SAP_ERR_UNSUPPORTED;
  int rc = ensure_device(nullptr);
  if (rc != SAP_OK) return rc;
  const int64_t n_rows = (row_end - row_begin) * n_q_heads;
  if (n_rows == 0) return SAP_OK;
  const int vec = head_dim / 4;
  const int group = (vec <= 32 && (vec & (vec - 1)) == 0) ? vec : 32;
  const int64_t want = (n_rows * group + kMergeThreads - 1) / kMergeThreads;
  const unsigned grid = static_cast<unsigned>(want < 148 * 16 ? want : 148 * 16);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (out_is_bf16)
    sap_lse_merge_kernel<true><<<grid, kMergeThreads, 0, st>>>(o_a, lse_a, o_b, lse_b, o_out, lse_out, n_tokens, n_q_heads, head_dim, row_begin, n_rows, group);
  else
    sap_lse_merge_kernel<false><<<grid, kMergeThreads, 0, st>>>(o_a, lse_a, o_b, lse_b, o_out, lse_out, n_tokens, n_q_heads, head_dim, row_begin, n_rows, group);
  g_launch_count.fetch_add(1);
  SAP_CUDA_CHECK(cudaGetLastError());
  return SAP_OK;
}

int sap_attn_bwd(const void* dout, const void* q, const void* k, const void* v, const void* out, const float* lse,
                 const int32_t* cu_seqlens_dev, sap_plan_t* plan, int64_t n_tokens, void* dq, void* dk, void* dv, int n_q_heads,
                 int n_kv_heads, int head_dim, float softmax_scale, void* workspace, size_t workspace_bytes,
                 void* cuda_stream) {
  if (!dout || !q || !k || !v || !out || !lse || !cu_seqlens_dev || !dq || !dk || !dv) return SAP_ERR_INVALID_ARG;
  int rc = check_call(plan, n_tokens, n_q_heads, n_kv_heads, head_dim, softmax_scale);
  if (rc != SAP_OK) return rc;
  if (!aligned16(dout) || !aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out) || !aligned16(dq) ||
      !aligned16(dk) || !aligned16(dv))
    return SAP_ERR_UNSUPPORTED;
  float *dsum, *dq_acc;
  if ((rc = bwd_ws(plan, n_q_heads, n_kv_heads, head_dim, workspace, workspace_bytes, &dsum, &dq_acc)) != SAP_OK) return rc;
  const PlanDevice* pd = static_cast<const PlanDevice*>(plan->dev_state);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (head_dim == 128)
    return launch_bwd<128>(pd, dout, q, k, v, out, lse, cu_seqlens_dev, plan, dq, dk, dv, n_q_heads, n_kv_heads,
                           softmax_scale, dsum, dq_acc, st);
  return launch_bwd<64>(pd, dout, q, k, v, out, lse, cu_seqlens_dev, plan, dq, dk, dv, n_q_heads, n_kv_heads,
                        softmax_scale, dsum, dq_acc, st);
}

int sap_attn_fwd_chunks(const void* q, const void* k, const void* v, const int32_t* cu_seqlens_dev, sap_plan_t* plan,
                        int64_t n_tokens, int32_t q_chunk_begin, int32_t q_chunk_end, void* out, float* lse, int n_q_heads,
                        int n_kv_heads, int head_dim, float softmax_scale, void* cuda_stream) {
  if (!q || !k || !v || !cu_seqlens_dev || !out || !lse) return SAP_ERR_INVALID_ARG;
  int rc = check_call(plan, n_tokens, n_q_heads, n_kv_heads, head_dim, softmax_scale);
  if (rc != SAP_OK) return rc;
  if (!chunk_range_ok(plan, q_chunk_begin, q_chunk_end)) return SAP_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out)) return SAP_ERR_UNSUPPORTED;
  if (q_chunk_begin == q_chunk_end) return SAP_OK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  RangeUse use, use2;
  if ((rc = use.acquire(plan, kRangeQ, q_chunk_begin, q_chunk_end, st)) != SAP_OK) return rc;
  const bool odd = (n_q_heads / n_kv_heads) % 2 != 0;   // odd Hq/Hkv (MHA): the row-pair form needs the same rows in 256-row tiles
  if (odd && (rc = use2.acquire(plan, kRangeQ2, q_chunk_begin, q_chunk_end, st)) != SAP_OK) return rc;
  const DevProgram &prog = use.prog, &prog2 = use2.prog;
  if (head_dim == 128)
    return launch_fwd<128, false>(prog, q, k, v, cu_seqlens_dev, plan, out, nullptr, lse, n_q_heads, n_kv_heads, softmax_scale, st, odd ? &prog2 : nullptr);
  return launch_fwd<64, false>(prog, q, k, v, cu_seqlens_dev, plan, out, nullptr, lse, n_q_heads, n_kv_heads, softmax_scale, st, odd ? &prog2 : nullptr);
}

int sap_attn_bwd_begin(const void* dout, const void* out, sap_plan_t* plan, int64_t n_tokens, int32_t q_chunk_begin,
                       int32_t q_chunk_end, int n_q_heads, int n_kv_heads, int head_dim, void* workspace,
                       size_t workspace_bytes, void* cuda_stream) {
  if (!dout || !out) return SAP_ERR_INVALID_ARG;
  int rc = check_call(plan, n_tokens, n_q_heads, n_kv_heads, head_dim, 1.f, /*need_upload=*/false);
  if (rc != SAP_OK) return rc;
  if (!chunk_range_ok(plan, q_chunk_begin, q_chunk_end)) return SAP_ERR_INVALID_ARG;
  if (!aligned16(dout) || !aligned16(out)) return SAP_ERR_UNSUPPORTED;
  float *dsum, *dq_acc;
  if ((rc = bwd_ws(plan, n_q_heads, n_kv_heads, head_dim, workspace, workspace_bytes, &dsum, &dq_acc)) != SAP_OK) return rc;
  const int64_t t0 = (int64_t)q_chunk_begin * plan->chunk_len, nt = (int64_t)(q_chunk_end - q_chunk_begin) * plan->chunk_len;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (head_dim == 128) return launch_bwd_pre<128>(dout, out, plan->n_tokens, n_q_heads, t0, nt, dsum, dq_acc, true, st);
  return launch_bwd_pre<64>(dout, out, plan->n_tokens, n_q_heads, t0, nt, dsum, dq_acc, true, st);
}

// shared tail of sap_attn_bwd_chunks / sap_attn_bwd_items
static int bwd_range(int kind1, int kind2, int32_t a, int32_t b, const void* dout, const void* q, const void* k, const void* v,
                     const float* lse, const int32_t* cu, sap_plan_t* plan, void* dk, void* dv, int Hq, int Hkv, int d,
                     float scale, void* workspace, size_t workspace_bytes, cudaStream_t st) {
  if (!aligned16(dout) || !aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(dk) || !aligned16(dv)) return SAP_ERR_UNSUPPORTED;
  float *dsum, *dq_acc;
  int rc;
  if ((rc = bwd_ws(plan, Hq, Hkv, d, workspace, workspace_bytes, &dsum, &dq_acc)) != SAP_OK) return rc;
  if (a == b) return SAP_OK;
  RangeUse use;
  if ((rc = use.acquire(plan, use_pair_kernel(d) ? kind2 : kind1, a, b, st)) != SAP_OK) return rc;
  const DevProgram& prog = use.prog;
  if (d == 128) return launch_bwd_main<128>(prog, prog, dout, q, k, v, lse, cu, plan, dk, dv, Hq, Hkv, scale, dsum, dq_acc, st);
  return launch_bwd_main<64>(prog, prog, dout, q, k, v, lse, cu, plan, dk, dv, Hq, Hkv, scale, dsum, dq_acc, st);
}

int sap_attn_bwd_chunks(const void* dout, const void* q, const void* k, const void* v, const float* lse,
                        const int32_t* cu_seqlens_dev, sap_plan_t* plan, int64_t n_tokens, int32_t kv_chunk_begin,
                        int32_t kv_chunk_end, void* dk, void* dv, int n_q_heads, int n_kv_heads, int head_dim,
                        float softmax_scale, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!dout || !q || !k || !v || !lse || !cu_seqlens_dev || !dk || !dv) return SAP_ERR_INVALID_ARG;
  int rc = check_call(plan, n_tokens, n_q_heads, n_kv_heads, head_dim, softmax_scale);
  if (rc != SAP_OK) return rc;
  if (!chunk_range_ok(plan, kv_chunk_begin, kv_chunk_end)) return SAP_ERR_INVALID_ARG;
  if (plan->chunk_len % kTile != 0) return SAP_ERR_UNSUPPORTED;  // K/V tiles must not straddle two ranks' chunks
  return bwd_range(kRangeKv, kRangeKvPair, kv_chunk_begin, kv_chunk_end, dout, q, k, v, lse, cu_seqlens_dev, plan, dk, dv,
                   n_q_heads, n_kv_heads, head_dim, softmax_scale, workspace, workspace_bytes, static_cast<cudaStream_t>(cuda_stream));
}

int sap_attn_bwd_items(const void* dout, const void* q, const void* k, const void* v, const float* lse,
                       const int32_t* cu_seqlens_dev, sap_plan_t* plan, int64_t n_tokens, int32_t item_begin,
                       int32_t item_end, void* dk, void* dv, int n_q_heads, int n_kv_heads, int head_dim,
                       float softmax_scale, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!dout || !q || !k || !v || !lse || !cu_seqlens_dev || !dk || !dv) return SAP_ERR_INVALID_ARG;
  int rc = check_call(plan, n_tokens, n_q_heads, n_kv_heads, head_dim, softmax_scale);
  if (rc != SAP_OK) return rc;
  if (!item_range_ok(plan, item_begin, item_end)) return SAP_ERR_INVALID_ARG;
  return bwd_range(kRangeItemsKv, kRangeItemsKvPair, item_begin, item_end, dout, q, k, v, lse, cu_seqlens_dev, plan, dk, dv,
                   n_q_heads, n_kv_heads, head_dim, softmax_scale, workspace, workspace_bytes, static_cast<cudaStream_t>(cuda_stream));
}

int sap_attn_bwd_end(sap_plan_t* plan, int64_t n_tokens, int32_t q_chunk_begin, int32_t q_chunk_end, void* dq, int n_q_heads,
                     int n_kv_heads, int head_dim, float softmax_scale, void* workspace, size_t workspace_bytes,
                     void* cuda_stream) {
  if (!dq) return SAP_ERR_INVALID_ARG;
  int rc = check_call(plan, n_tokens, n_q_heads, n_kv_heads, head_dim, softmax_scale, /*need_upload=*/false);
  if (rc != SAP_OK) return rc;
  if (!chunk_range_ok(plan, q_chunk_begin, q_chunk_end)) return SAP_ERR_INVALID_ARG;
  if (!aligned16(dq)) return SAP_ERR_UNSUPPORTED;
  float *dsum, *dq_acc;
  if ((rc = bwd_ws(plan, n_q_heads, n_kv_heads, head_dim, workspace, workspace_bytes, &dsum, &dq_acc)) != SAP_OK) return rc;
  const int64_t t0 = (int64_t)q_chunk_begin * plan->chunk_len, nt = (int64_t)(q_chunk_end - q_chunk_begin) * plan->chunk_len;
  return launch_bwd_post(dq_acc, dq, n_q_heads, head_dim, t0, nt, softmax_scale, static_cast<cudaStream_t>(cuda_stream));
}

int sap_axpy(void* dst, int dst_is_bf16, const void* src, int src_is_bf16, int64_t n_elems, float alpha, int accumulate,
             void* cuda_stream) {
  if (!dst || !src || n_elems < 0) return SAP_ERR_INVALID_ARG;
  if (n_elems % 8 != 0 || !aligned16(dst) || !aligned16(src)) return SAP_ERR_UNSUPPORTED;
  int rc = ensure_device(nullptr);
  if (rc != SAP_OK) return rc;
  if (n_elems == 0) return SAP_OK;
  const int64_t n8 = n_elems / 8, want = (n8 + 255) / 256;
  const unsigned grid = static_cast<unsigned>(want < 148 * 16 ? want : 148 * 16);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (dst_is_bf16 && src_is_bf16) sap_axpy_kernel<true, true><<<grid, 256, 0, st>>>(dst, src, n8, alpha, accumulate);
  else if (dst_is_bf16) sap_axpy_kernel<true, false><<<grid, 256, 0, st>>>(dst, src, n8, alpha, accumulate);
  else if (src_is_bf16) sap_axpy_kernel<false, true><<<grid, 256, 0, st>>>(dst, src, n8, alpha, accumulate);
  else sap_axpy_kernel<false, false><<<grid, 256, 0, st>>>(dst, src, n8, alpha, accumulate);
  g_launch_count.fetch_add(1);
  SAP_CUDA_CHECK(cudaGetLastError());
  return SAP_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// sap_attn_bwd_static (include/sap.h): the backward pass for callers that must not allocate device memory.
//
// sap_attn_bwd needs two pieces of device memory besides its tensors: the plan's tile programs (sap_plan_upload:
// cudaMalloc + a synchronous copy) and the caller's workspace (D and the fp32 dQ accumulator).  Here both live in one
// file-scope device array that comes with the library image: nobody allocates it and nobody frees it.
//
//   g_static_scratch = [ tile program: tiles | segs    (kStaticProgramBytes)
//                      | workspace: D [Hq,N] fp32 | dQ accumulator [N,Hq,d] fp32   (SAP_STATIC_WORKSPACE_BYTES) ]
//
// In host code the identifier g_static_scratch is only the host-side handle of the symbol - it is not a device
// address and must never reach a kernel or a memcpy as one.  The device address is looked up once per device with
// cudaGetSymbolAddress (below, with that device current) and everything on the host works from that pointer.
// ---------------------------------------------------------------------------------------------------------------------
namespace sap {

constexpr size_t kStaticProgramBytes = size_t(256) << 10;   // far more than any plan whose workspace fits below needs
static __device__ __align__(256) unsigned char g_static_scratch[kStaticProgramBytes + SAP_STATIC_WORKSPACE_BYTES];

static unsigned char* g_static_base[64];   // device address of g_static_scratch per device; null = not set up yet
static std::mutex g_static_mu;

// Set-up of the current device for sap_attn_bwd_static, on its first call there: architecture check, the kernels'
// shared-memory opt-ins, the address of the scratch array.  Unlike ensure_device it allocates nothing (that one also
// creates the forward's counter pool with cudaMalloc), so the two are kept apart.
static int ensure_device_static(unsigned char** base) {
  int dev = 0;
  SAP_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return SAP_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_base[dev]) {
    int major = 0;
    SAP_CUDA_CHECK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return SAP_ERR_WRONG_ARCH;
    const cudaFuncAttribute a = cudaFuncAttributeMaxDynamicSharedMemorySize;
    SAP_CUDA_CHECK(cudaFuncSetAttribute(sap_bwd_fused_kernel<64>, a, FusedSmem<64>::kTotal));
    SAP_CUDA_CHECK(cudaFuncSetAttribute(sap_bwd_fused_kernel<128>, a, FusedSmem<128>::kTotal));
    SAP_CUDA_CHECK(cudaFuncSetAttribute(sap_bwd_pair_kernel, a, PairSmem::kTotal));
    void* p = nullptr;
    SAP_CUDA_CHECK(cudaGetSymbolAddress(&p, g_static_scratch));
    if (!p) { g_last_cuda_error = static_cast<int>(cudaErrorInvalidSymbol); return SAP_ERR_CUDA; }
    g_static_base[dev] = static_cast<unsigned char*>(p);
  }
  *base = g_static_base[dev];
  return SAP_OK;
}

}  // namespace sap

extern "C" int sap_attn_bwd_static(const void* dout, const void* q, const void* k, const void* v, const void* out,
                                   const float* lse, const int32_t* cu_seqlens_dev, sap_plan_t* plan, int64_t n_tokens,
                                   void* dq, void* dk, void* dv, int n_q_heads, int n_kv_heads, int head_dim,
                                   float softmax_scale, void* cuda_stream) {
  if (!dout || !q || !k || !v || !out || !lse || !cu_seqlens_dev || !dq || !dk || !dv || !plan) return SAP_ERR_INVALID_ARG;
  if (n_q_heads < 1 || n_kv_heads < 1 || !(softmax_scale > 0.f)) return SAP_ERR_INVALID_ARG;
  if ((head_dim != 64 && head_dim != 128) || n_q_heads % n_kv_heads != 0) return SAP_ERR_UNSUPPORTED;
  if (n_tokens != plan->n_tokens) return SAP_ERR_PLAN_MISMATCH;
  if (!aligned16(dout) || !aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out) || !aligned16(dq) ||
      !aligned16(dk) || !aligned16(dv))
    return SAP_ERR_UNSUPPORTED;
  if (g_bwd_stages.load() != kBwdDefaultStages) return SAP_ERR_UNSUPPORTED;   // the diagnostic split forms walk other programs
  // the limits, checked before anything touches the device
  const TileProgram& host = use_pair_kernel(head_dim) ? plan->kv2 : plan->kv;   // the program the main kernel walks
  const size_t tiles_bytes = align256(host.tiles.size() * sizeof(TileDesc));
  const size_t segs_bytes = (host.segs.size() + 1) * sizeof(SegDesc);            // the kernels read one descriptor ahead
  if (tiles_bytes + segs_bytes > kStaticProgramBytes) return SAP_ERR_STATIC_LIMIT;
  if (sap_workspace_bytes(plan, n_q_heads, n_kv_heads, head_dim, SAP_PASS_BWD) > SAP_STATIC_WORKSPACE_BYTES) return SAP_ERR_STATIC_LIMIT;
  unsigned char* base = nullptr;
  int rc = ensure_device_static(&base);
  if (rc != SAP_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  // This call's tile program goes into the scratch array on the caller's stream, in front of the kernels that read it.
  // The source is the plan's host copy, which lives as long as the plan.
  PlanDevice pd;
  DevProgram prog;
  prog.tiles = reinterpret_cast<TileDesc*>(base);
  prog.segs = reinterpret_cast<SegDesc*>(base + tiles_bytes);
  prog.n_tiles = static_cast<int32_t>(host.tiles.size());
  if (!host.tiles.empty())
    SAP_CUDA_CHECK(cudaMemcpyAsync(prog.tiles, host.tiles.data(), host.tiles.size() * sizeof(TileDesc), cudaMemcpyHostToDevice, st));
  if (!host.segs.empty())
    SAP_CUDA_CHECK(cudaMemcpyAsync(prog.segs, host.segs.data(), host.segs.size() * sizeof(SegDesc), cudaMemcpyHostToDevice, st));
  pd.kv = pd.kv2 = prog;     // launch_bwd_main reads the one that matches the kernel it picks
  // The workspace half: D is overwritten in full by the pre-pass; the accumulator still holds the previous call's sums
  // and is cleared by launch_bwd (cudaMemsetAsync on the stream) in front of the main kernel.
  float* dsum = reinterpret_cast<float*>(base + kStaticProgramBytes);
  float* dq_acc = reinterpret_cast<float*>(base + kStaticProgramBytes + align256(static_cast<size_t>(plan->n_tokens) * n_q_heads * sizeof(float)));
  if (head_dim == 128)
    return launch_bwd<128>(&pd, dout, q, k, v, out, lse, cu_seqlens_dev, plan, dq, dk, dv, n_q_heads, n_kv_heads,
                           softmax_scale, dsum, dq_acc, st);
  return launch_bwd<64>(&pd, dout, q, k, v, out, lse, cu_seqlens_dev, plan, dq, dk, dv, n_q_heads, n_kv_heads,
                        softmax_scale, dsum, dq_acc, st);
}
