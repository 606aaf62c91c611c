// Internal structures shared by the host planner and the kernels (not part of the C ABI).
#pragma once
#include <stdint.h>
#include <mutex>
#include <vector>
#include "../../include/sap.h"

namespace sap {

constexpr int kTile = 128;  // rows of a Q tile and of a K/V tile

// One stationary tile of a kernel: a Q tile (fwd, bwd-dQ) or a K/V tile (bwd-dKdV).
struct TileDesc {
  int32_t row0;       // first token of the tile
  int32_t rows;       // valid tokens (1..128; 1..256 for the K/V pair-tiles of sap_bwd_pair_kernel and the row-pair Q tiles)
  int32_t seg_begin;  // segments [seg_begin, seg_end) of the matching SegDesc array
  int32_t seg_end;
};

// One run of streamed tiles that belongs to one plan item.  The streamed tiles start at
// t_begin (a multiple of 128), step 128, while < t_end.  Mask of element (row t, key s):
//   visible iff  q_lo <= t < q_hi  and  kv_lo <= s < kv_hi  and  same document  and  s <= t.
struct SegDesc {
  int32_t t_begin, t_end;
  int32_t q_lo, q_hi;
  int32_t kv_lo, kv_hi;
  int32_t item;   // index into sap_plan_items
  int32_t pad;
};

struct TileProgram {
  std::vector<TileDesc> tiles;  // launch order: Q-stationary longest first; KV-stationary by document, longest first inside
  std::vector<SegDesc> segs;
  int64_t streamed_tiles = 0;   // total streamed 128x128 tiles (per head)
};

}  // namespace sap

struct sap_plan {
  int32_t n_docs = 0, n_chunks = 0, n_tokens = 0, chunk_len = 0;
  std::vector<int32_t> cu;
  std::vector<sap_item_t> items;
  std::vector<int32_t> chunk_offsets, kv_offsets, kv_index;
  std::vector<uint8_t> kind_map;
  int64_t useful_pairs = 0;
  sap::TileProgram fwd;  // Q-stationary: forward and backward-dQ
  sap::TileProgram fwd2; // Q-stationary, 256-row tiles = two 128-row units of one head (row-pair forward: odd Hq/Hkv, MHA)
  sap::TileProgram kv;   // KV-stationary: backward-dK/dV, 128-key tiles (one CTA per tile)
  sap::TileProgram kv2;  // KV-stationary, 256-key pair-tiles (one CTA pair per tile)
  std::mutex mu;
  void* dev_state = nullptr;  // sap::PlanDevice*, created by sap_plan_upload (CUDA half of the library)
};

namespace sap {
// Build a Q-stationary tile program restricted to items [item_begin, item_end).
// `drop_empty`: leave out tiles that have no work among those items (a rank's launch touches only its own rows).
void build_q_program(const sap_plan& p, int32_t item_begin, int32_t item_end, TileProgram& out, bool drop_empty = false,
                     int32_t tile_rows = kTile);
// K/V tiles of kv-chunks [chunk_begin, chunk_end) only (the whole sequence by default).
// `item_begin..item_end` keeps only segments of those plan items; `drop_empty` leaves out tiles without work.
void build_kv_program(const sap_plan& p, TileProgram& out, int32_t chunk_begin = 0, int32_t chunk_end = -1, int32_t tile_rows = kTile,
                      int32_t item_begin = 0, int32_t item_end = -1, bool drop_empty = false);
}  // namespace sap
