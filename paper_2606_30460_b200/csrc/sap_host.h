// Host-side helpers of the CUDA half of the library: error bookkeeping, tensor-map encoding,
// device mirrors of the tile programs.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <atomic>
#include <list>
#include <utility>
#include <vector>
#include "sap_internal.h"

namespace sap {

extern thread_local int g_last_cuda_error;
extern std::atomic<int64_t> g_launch_count;

#define SAP_CUDA_CHECK(expr)                                   \
  do {                                                         \
    cudaError_t _e = (expr);                                   \
    if (_e != cudaSuccess) {                                   \
      sap::g_last_cuda_error = static_cast<int>(_e);           \
      return (_e == cudaErrorNoDevice || _e == cudaErrorInsufficientDriver) ? SAP_ERR_NO_DEVICE : SAP_ERR_CUDA; \
    }                                                          \
  } while (0)

struct DevProgram {
  TileDesc* tiles = nullptr;
  SegDesc* segs = nullptr;
  int32_t n_tiles = 0;
};

// A range-restricted program (partial forward over an item range, per-rank launches over a chunk range, per-item
// backward): built on first use, uploaded on the caller's stream, kept with the plan.
struct RangeProgram {
  std::pair<int32_t, int32_t> key;
  TileProgram host;            // source of the asynchronous upload; must outlive it
  DevProgram dev;
  cudaEvent_t ready = nullptr; // recorded behind the upload: other streams wait on it
  cudaStream_t stream = nullptr;
  // Life time (sap_api.cu: RangeUse): a call pins the entry from lookup until its kernels are enqueued and then records
  // an event behind them on its stream; eviction takes only unpinned entries and frees their memory behind all of
  // those events.  An entry a CUDA graph has recorded a launch on stays until sap_plan_destroy.
  int pins = 0;
  bool held_by_graph = false;
  std::vector<std::pair<cudaStream_t, cudaEvent_t>> used;   // last use per stream that ran kernels on this program
};
enum { kRangeItemsQ = 0, kRangeQ = 1, kRangeKv = 2, kRangeKvPair = 3, kRangeItemsKv = 4, kRangeItemsKvPair = 5, kRangeItemsQDrop = 6, kRangeQ2 = 7, kRangeKinds = 8 };

// Device copies owned by a plan (freed by sap_plan_destroy).  A plan's mirror lives on ONE device (the current
// device of the first upload); calls with another current device return SAP_ERR_PLAN_MISMATCH.
struct PlanDevice {
  bool uploaded = false;
  int device = -1;
  DevProgram fwd, kv, kv2, fwd2;
  std::list<RangeProgram> ranges[kRangeKinds];   // most recently used first
};

int ensure_device(int* dev_out);
int upload_program(const TileProgram& host, DevProgram& dev);
void free_program(DevProgram& dev);

// 2D bf16 tensor map over a [n_rows, n_heads*head_dim] matrix, box = 64 columns x box_rows rows, 128-byte swizzle.
int make_tile_map(CUtensorMap* map, const void* base, int64_t n_rows, int64_t row_elems, int box_rows = kTile);

}  // namespace sap
