// Host-side JIT planner (§3.1-3.2: "compile" side of SAP's compile-execute split, :75,:106-:120).
//
// Step 1 of the paper's compiler partitions the attention mask by rank rows/columns and classifies
// each (q_chunk, kv_chunk) block (:108).  With contiguous equal chunks (n = N/P, :59) and the cu_len
// visibility rule (:45) the classification has a closed form, used here (the oracle's planner instead
// loops over all documents for every pair):
//   * j == i : DIAG.  Rows = keys = the whole chunk; documents doc(i*n) .. doc((i+1)*n - 1).
//   * j <  i : at most one document can reach back into chunk j: e* = doc(i*n), and it does iff
//              cu[e*] < (j+1)*n.  Rows [i*n, min(cu[e*+1], (i+1)*n)), keys [max(cu[e*], j*n), (j+1)*n);
//              every (row, key) of that rectangle is visible => FULL needs no mask.
// doc(t) = the unique e with cu[e] <= t < cu[e+1] (zero-length documents never contain a token).
//
// The planner then "jits" the item lists into per-tile programs (TileDesc/SegDesc) the kernels walk:
// the analogue of the paper's per-rank instruction lists (:120), at 128-row tile granularity.
#include <algorithm>
#include <cstring>
#include <new>
#include "sap_internal.h"

namespace sap {

static inline int32_t doc_of(const std::vector<int32_t>& cu, int64_t t) {
  // last e with cu[e] <= t  (upper_bound - 1); skips zero-length documents automatically
  return (int32_t)(std::upper_bound(cu.begin(), cu.end(), (int32_t)t) - cu.begin()) - 1;
}

static inline int32_t floor_tile(int64_t x) { return (int32_t)(x / kTile * kTile); }

// Launch order of a program's tiles.  Tiles of one `group` (a document) stream the same rows or keys: keeping them
// adjacent keeps what they share - for the KV-stationary programs the document's part of the fp32 dQ accumulator and its
// Q / dO rows, for the Q-stationary program the document's K / V - in L2 while it is live.  Documents longest first and,
// inside a document, longest tile first (LPT), so that a launch still ends on short tiles.
constexpr int32_t kGroupQTilesFromTokens = 192 * 1024;

static void order_tiles(TileProgram& out, const std::vector<int64_t>& work, const std::vector<int32_t>& group, int32_t n_docs) {
  std::vector<int64_t> group_work(n_docs, 0);
  for (size_t k = 0; k < work.size(); ++k) group_work[group[k]] = std::max(group_work[group[k]], work[k]);
  std::vector<int32_t> order(out.tiles.size());
  for (size_t k = 0; k < order.size(); ++k) order[k] = (int32_t)k;
  std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) {
    if (group[a] != group[b]) {
      if (group_work[group[a]] != group_work[group[b]]) return group_work[group[a]] > group_work[group[b]];
      return group[a] < group[b];
    }
    return work[a] > work[b];
  });
  std::vector<TileDesc> sorted(out.tiles.size());
  for (size_t k = 0; k < order.size(); ++k) sorted[k] = out.tiles[order[k]];
  out.tiles.swap(sorted);
}

void build_q_program(const sap_plan& p, int32_t item_begin, int32_t item_end, TileProgram& out, bool drop_empty, int32_t tile_rows) {
  out.tiles.clear();
  out.segs.clear();
  out.streamed_tiles = 0;
  const int64_t n = p.chunk_len;
  std::vector<int64_t> work;
  std::vector<int32_t> group;
  for (int32_t i = 0; i < p.n_chunks; ++i) {
    const int64_t c_begin = (int64_t)i * n, c_end = c_begin + n;
    for (int64_t r0 = c_begin; r0 < c_end; r0 += tile_rows) {   // 128 rows; 256 = two 128-row units of the row-pair forward
      const int64_t r1 = std::min<int64_t>(r0 + tile_rows, c_end);
      TileDesc td;
      td.row0 = (int32_t)r0;
      td.rows = (int32_t)(r1 - r0);
      td.seg_begin = (int32_t)out.segs.size();
      int64_t w = 0;
      for (int32_t it = p.chunk_offsets[i]; it < p.chunk_offsets[i + 1]; ++it) {
        if (it < item_begin || it >= item_end) continue;
        const sap_item_t& im = p.items[it];
        const int64_t ra = std::max<int64_t>(r0, im.q_begin), rb = std::min<int64_t>(r1, im.q_end);
        if (ra >= rb) continue;
        // keys needed by rows [ra, rb): from the start of the first row's document up to the last row
        const int64_t lo = std::max<int64_t>(im.kv_begin, p.cu[doc_of(p.cu, ra)]);
        const int64_t hi = std::min<int64_t>(im.kv_end, rb);
        if (lo >= hi) continue;
        SegDesc sd;
        sd.t_begin = floor_tile(lo);
        sd.t_end = (int32_t)hi;
        sd.q_lo = im.q_begin; sd.q_hi = im.q_end;
        sd.kv_lo = im.kv_begin; sd.kv_hi = im.kv_end;
        sd.item = it; sd.pad = 0;
        out.segs.push_back(sd);
        w += (hi - sd.t_begin + kTile - 1) / kTile;
      }
      td.seg_end = (int32_t)out.segs.size();
      if (drop_empty && td.seg_end == td.seg_begin) continue;
      out.tiles.push_back(td);
      work.push_back(w);
      group.push_back(doc_of(p.cu, r0));
      out.streamed_tiles += w;
    }
  }
  // group = the document of the tile's first row (the longest key stream).  Grouping pays once one kv-head's K and V
  // (512 B per token at head_dim 128) no longer fit in L2 beside everything else: measured on a B200, cfg5 (512K tokens)
  // 32.6 -> 11.3 GB of DRAM traffic per launch and 1 % less time, cfg3 (128K) no change, cfg2 (32K) 1.7 % MORE time than
  // plain longest-first.  Below the threshold all tiles form one group, i.e. plain LPT.
  if (p.n_tokens < kGroupQTilesFromTokens) std::fill(group.begin(), group.end(), 0);
  order_tiles(out, work, group, p.n_docs);
}

void build_kv_program(const sap_plan& p, TileProgram& out, int32_t chunk_begin, int32_t chunk_end, int32_t tile_rows,
                      int32_t item_begin, int32_t item_end, bool drop_empty) {
  if (item_end < 0) item_end = (int32_t)p.items.size();
  out.tiles.clear();
  out.segs.clear();
  out.streamed_tiles = 0;
  const int64_t n = p.chunk_len, N = p.n_tokens;
  std::vector<int64_t> work;
  std::vector<int32_t> group;
  // K/V tiles of `tile_rows` keys (128: one CTA; 256: a CTA pair) counted from the first key of the range (they must
  // match the key tiles the forward kernel streams only in coverage, not in alignment); a tile that straddles two
  // kv-chunks gets segments from both.
  const int64_t k_begin = (int64_t)chunk_begin * n, k_end = chunk_end < 0 ? N : (int64_t)chunk_end * n;  // 128-aligned when restricted
  for (int64_t c0 = k_begin; c0 < k_end; c0 += tile_rows) {
    const int64_t c1 = std::min<int64_t>(c0 + tile_rows, k_end);
    TileDesc td;
    td.row0 = (int32_t)c0;
    td.rows = (int32_t)(c1 - c0);
    td.seg_begin = (int32_t)out.segs.size();
    int64_t w = 0;
    const int32_t j_lo = (int32_t)(c0 / n), j_hi = (int32_t)((c1 - 1) / n);
    for (int32_t j = j_lo; j <= j_hi; ++j) {
      for (int32_t x = p.kv_offsets[j]; x < p.kv_offsets[j + 1]; ++x) {
        const int32_t it = p.kv_index[x];
        if (it < item_begin || it >= item_end) continue;
        const sap_item_t& im = p.items[it];
        const int64_t ca = std::max<int64_t>(c0, im.kv_begin), cb = std::min<int64_t>(c1, im.kv_end);
        if (ca >= cb) continue;
        // rows that see keys [ca, cb): from the first key up to the end of the last key's document
        const int64_t lo = std::max<int64_t>(im.q_begin, ca);
        const int64_t hi = std::min<int64_t>(im.q_end, p.cu[doc_of(p.cu, cb - 1) + 1]);
        if (lo >= hi) continue;
        SegDesc sd;
        sd.t_begin = floor_tile(lo);
        sd.t_end = (int32_t)hi;
        sd.q_lo = im.q_begin; sd.q_hi = im.q_end;
        sd.kv_lo = im.kv_begin; sd.kv_hi = im.kv_end;
        sd.item = it; sd.pad = 0;
        out.segs.push_back(sd);
        w += (hi - sd.t_begin + kTile - 1) / kTile;
      }
    }
    td.seg_end = (int32_t)out.segs.size();
    if (drop_empty && td.seg_end == td.seg_begin) continue;
    out.tiles.push_back(td);
    work.push_back(w);
    group.push_back(doc_of(p.cu, c1 - 1));
    out.streamed_tiles += w;
  }
  order_tiles(out, work, group, p.n_docs);   // group = the document of the tile's last key (whose tail the tile streams)
}

}  // namespace sap

using namespace sap;

extern "C" {

int sap_plan_create(const int32_t* cu, int32_t n_docs, int32_t n_chunks, sap_plan_t** out) {
  if (!cu || !out || n_docs < 1 || n_chunks < 1) return SAP_ERR_INVALID_ARG;
  if (cu[0] != 0) return SAP_ERR_BAD_CU_SEQLENS;
  for (int32_t e = 0; e < n_docs; ++e)
    if (cu[e + 1] < cu[e]) return SAP_ERR_BAD_CU_SEQLENS;
  const int64_t N = cu[n_docs];
  if (N <= 0) return SAP_ERR_BAD_CU_SEQLENS;
  const int32_t P = n_chunks;
  if (N % P != 0) return SAP_ERR_INDIVISIBLE;
  sap_plan* p = new (std::nothrow) sap_plan();
  if (!p) return SAP_ERR_INVALID_ARG;
  p->n_docs = n_docs; p->n_chunks = P; p->n_tokens = (int32_t)N; p->chunk_len = (int32_t)(N / P);
  p->cu.assign(cu, cu + n_docs + 1);
  const int64_t n = p->chunk_len;
  p->kind_map.assign((size_t)P * P, (uint8_t)SAP_MASK_SKIP);
  p->chunk_offsets.resize(P + 1);
  for (int32_t i = 0; i < P; ++i) {
    p->chunk_offsets[i] = (int32_t)p->items.size();
    const int64_t r_begin = (int64_t)i * n, r_end = r_begin + n;
    const int32_t e_first = doc_of(p->cu, r_begin), e_last = doc_of(p->cu, r_end - 1);
    {  // step 0: the diagonal block
      sap_item_t im;
      im.q_chunk = i; im.kv_chunk = i; im.doc_lo = e_first; im.doc_hi = e_last;
      im.mask_kind = SAP_MASK_DIAG; im.step = 0;
      im.q_begin = (int32_t)r_begin; im.q_end = (int32_t)r_end;
      im.kv_begin = (int32_t)r_begin; im.kv_end = (int32_t)r_end;
      p->items.push_back(im);
      p->kind_map[(size_t)i * P + i] = (uint8_t)SAP_MASK_DIAG;
    }
    const int64_t d_begin = p->cu[e_first], d_end = p->cu[e_first + 1];
    for (int32_t s = 1; s <= i; ++s) {  // ring order: j = i-1, i-2, ...
      const int32_t j = i - s;
      if (d_begin >= (int64_t)(j + 1) * n) break;  // the document does not reach chunk j (nor any earlier one)
      sap_item_t im;
      im.q_chunk = i; im.kv_chunk = j; im.doc_lo = e_first; im.doc_hi = e_first;
      im.mask_kind = SAP_MASK_FULL; im.step = s;
      im.q_begin = (int32_t)r_begin; im.q_end = (int32_t)std::min<int64_t>(d_end, r_end);
      im.kv_begin = (int32_t)std::max<int64_t>(d_begin, (int64_t)j * n); im.kv_end = (int32_t)((int64_t)(j + 1) * n);
      p->items.push_back(im);
      p->kind_map[(size_t)i * P + j] = (uint8_t)SAP_MASK_FULL;
    }
  }
  p->chunk_offsets[P] = (int32_t)p->items.size();
  // transposed index (CSR by kv_chunk, item ids ascending) for the backward pass
  p->kv_offsets.assign(P + 1, 0);
  for (const sap_item_t& im : p->items) p->kv_offsets[im.kv_chunk + 1]++;
  for (int32_t j = 0; j < P; ++j) p->kv_offsets[j + 1] += p->kv_offsets[j];
  p->kv_index.resize(p->items.size());
  {
    std::vector<int32_t> fill(p->kv_offsets.begin(), p->kv_offsets.end() - 1);
    for (int32_t it = 0; it < (int32_t)p->items.size(); ++it) p->kv_index[fill[p->items[it].kv_chunk]++] = it;
  }
  for (int32_t e = 0; e < n_docs; ++e) {
    const int64_t L = (int64_t)cu[e + 1] - cu[e];
    p->useful_pairs += L * (L + 1) / 2;
  }
  build_q_program(*p, 0, (int32_t)p->items.size(), p->fwd);
  build_q_program(*p, 0, (int32_t)p->items.size(), p->fwd2, false, 2 * kTile);
  build_kv_program(*p, p->kv);
  build_kv_program(*p, p->kv2, 0, -1, 2 * kTile);
  *out = p;
  return SAP_OK;
}

int32_t sap_plan_n_items(const sap_plan_t* p) { return p ? (int32_t)p->items.size() : 0; }
int32_t sap_plan_n_chunks(const sap_plan_t* p) { return p ? p->n_chunks : 0; }
int32_t sap_plan_n_tokens(const sap_plan_t* p) { return p ? p->n_tokens : 0; }
const sap_item_t* sap_plan_items(const sap_plan_t* p) { return p ? p->items.data() : nullptr; }
const int32_t* sap_plan_chunk_offsets(const sap_plan_t* p) { return p ? p->chunk_offsets.data() : nullptr; }
const int32_t* sap_plan_kv_offsets(const sap_plan_t* p) { return p ? p->kv_offsets.data() : nullptr; }
const int32_t* sap_plan_kv_index(const sap_plan_t* p) { return p ? p->kv_index.data() : nullptr; }
const uint8_t* sap_plan_kind_map(const sap_plan_t* p) { return p ? p->kind_map.data() : nullptr; }
int64_t sap_plan_useful_pairs(const sap_plan_t* p) { return p ? p->useful_pairs : 0; }
int64_t sap_plan_fwd_tiles(const sap_plan_t* p) { return p ? p->fwd.streamed_tiles : 0; }

int sap_plan_schedule(const sap_plan_t* p, int32_t policy, sap_slot_t* slots, int32_t* n_stages) {
  if (!p || !slots || !n_stages || (policy != SAP_SCHED_RING && policy != SAP_SCHED_BALANCED)) return SAP_ERR_INVALID_ARG;
  const int32_t P = p->n_chunks, n_items = (int32_t)p->items.size();
  const int64_t n = p->chunk_len;
  int32_t last = 0;
  if (policy == SAP_SCHED_RING) {
    for (int32_t x = 0; x < n_items; ++x) {
      slots[x].rank = p->items[x].q_chunk;
      slots[x].stage = p->items[x].step;
      last = std::max(last, slots[x].stage);
    }
    *n_stages = last + 1;
    return SAP_OK;
  }
  // Step 2: regional strategy.  The region of a FULL item is its (single) document; it spans chunks a..b.
  std::vector<int32_t> regional(n_items);
  for (int32_t x = 0; x < n_items; ++x) {
    const sap_item_t& im = p->items[x];
    if (im.mask_kind == SAP_MASK_DIAG) { slots[x].rank = im.q_chunk; regional[x] = 0; continue; }
    const int32_t e = im.doc_lo;
    const int32_t a = (int32_t)(p->cu[e] / n), b = (int32_t)((p->cu[e + 1] - 1) / n), m = b - a + 1;
    const int32_t t = im.q_chunk - im.kv_chunk;
    if (t <= m / 2) { slots[x].rank = im.q_chunk; regional[x] = t; }
    else            { slots[x].rank = im.kv_chunk; regional[x] = m - t; }
  }
  // Step 3a: global balance.  While the busiest rank (lowest index on ties) holds a FULL item whose other end is at
  // least two items less loaded, hand over the one whose other end is least loaded (lowest item index on ties).
  std::vector<int32_t> load(P, 0), dist_of(n_items, 0), span_of(n_items, 0);
  for (int32_t x = 0; x < n_items; ++x) {
    ++load[slots[x].rank];
    const sap_item_t& im = p->items[x];
    if (im.mask_kind == SAP_MASK_DIAG) continue;
    const int32_t e = im.doc_lo;
    span_of[x] = (int32_t)((p->cu[e + 1] - 1) / n) - (int32_t)(p->cu[e] / n) + 1;
    dist_of[x] = im.q_chunk - im.kv_chunk;
  }
  for (;;) {
    int32_t R = 0;
    for (int32_t r = 1; r < P; ++r) if (load[r] > load[R]) R = r;
    int32_t best = -1, best_other = -1;
    for (int32_t x = 0; x < n_items; ++x) {
      const sap_item_t& im = p->items[x];
      if (slots[x].rank != R || im.mask_kind == SAP_MASK_DIAG) continue;
      const int32_t other = (R == im.q_chunk) ? im.kv_chunk : im.q_chunk;
      if (best < 0 || load[other] < load[best_other]) { best = x; best_other = other; }
    }
    if (best < 0 || load[best_other] + 1 >= load[R]) break;
    --load[R]; ++load[best_other];
    slots[best].rank = best_other;
    regional[best] = (best_other == p->items[best].q_chunk) ? dist_of[best] : span_of[best] - dist_of[best];
  }
  // Step 3b: one item per rank per stage: every rank runs its items in order of (regional stage, q_chunk, kv_chunk)
  std::vector<int32_t> order(n_items);
  for (int32_t x = 0; x < n_items; ++x) order[x] = x;
  std::stable_sort(order.begin(), order.end(), [&](int32_t x, int32_t y) {
    if (regional[x] != regional[y]) return regional[x] < regional[y];
    if (p->items[x].q_chunk != p->items[y].q_chunk) return p->items[x].q_chunk < p->items[y].q_chunk;
    return p->items[x].kv_chunk < p->items[y].kv_chunk;
  });
  std::vector<int32_t> next_stage(P, 0);  // a rank runs its items back to back: stage = position in its sorted list
  for (int32_t x : order) {
    slots[x].stage = next_stage[slots[x].rank]++;
    last = std::max(last, slots[x].stage);
  }
  *n_stages = last + 1;
  return SAP_OK;
}

// order inside a rank's list: stage; SEND / RECV by (opcode, tensor, peer, item), COMPUTING, COPY by (tensor, peer, item)
static int32_t emit_codes(std::vector<sap_code_t>& out, sap_code_t* codes, int32_t cap) {
  auto phase = [](const sap_code_t& c) { return c.opcode <= SAP_OP_RECV ? 0 : (c.opcode == SAP_OP_COMPUTING ? 1 : 2); };
  std::stable_sort(out.begin(), out.end(), [&](const sap_code_t& a, const sap_code_t& b) {
    if (a.stage != b.stage) return a.stage < b.stage;
    if (phase(a) != phase(b)) return phase(a) < phase(b);
    if (phase(a) == 0 && a.opcode != b.opcode) return a.opcode < b.opcode;
    if (a.tensor != b.tensor) return a.tensor < b.tensor;
    if (a.peer != b.peer) return a.peer < b.peer;
    return a.item < b.item;
  });
  const int32_t n = (int32_t)out.size();
  for (int32_t c = 0; c < n && c < cap; ++c) codes[c] = out[c];
  return n;
}

int32_t sap_plan_codegen(const sap_plan_t* p, const sap_slot_t* slots, int32_t rank, sap_code_t* codes, int32_t cap) {
  if (!p || !slots || rank < 0 || rank >= p->n_chunks || cap < 0 || (cap > 0 && !codes)) return -SAP_ERR_INVALID_ARG;
  const int32_t n_items = (int32_t)p->items.size();
  std::vector<sap_code_t> out;
  for (int32_t x = 0; x < n_items; ++x) {
    const sap_item_t& im = p->items[x];
    const int32_t i = im.q_chunk, j = im.kv_chunk, R = slots[x].rank, st = slots[x].stage;
    if (R != i && R != j) return -SAP_ERR_INVALID_ARG;
    if (R == rank) out.push_back({st, SAP_OP_COMPUTING, -1, -1, x});
    if (i == j) continue;
    if (R == i) {  // K/V_j travels j -> i one stage earlier
      if (rank == j) out.push_back({st - 1, SAP_OP_SEND, SAP_T_KV, i, x});
      if (rank == i) { out.push_back({st - 1, SAP_OP_RECV, SAP_T_KV, j, x}); out.push_back({st - 1, SAP_OP_COPY, SAP_T_KV, j, x}); }
    } else {       // helper: Q_i travels i -> j one stage earlier, the partial result j -> i one stage later
      if (rank == i) out.push_back({st - 1, SAP_OP_SEND, SAP_T_Q, j, x});
      if (rank == j) { out.push_back({st - 1, SAP_OP_RECV, SAP_T_Q, i, x}); out.push_back({st - 1, SAP_OP_COPY, SAP_T_Q, i, x}); }
      if (rank == j) out.push_back({st + 1, SAP_OP_SEND, SAP_T_O, i, x});
      if (rank == i) { out.push_back({st + 1, SAP_OP_RECV, SAP_T_O, j, x}); out.push_back({st + 1, SAP_OP_COPY, SAP_T_O, j, x}); }
    }
  }
  return emit_codes(out, codes, cap);
}

int32_t sap_plan_codegen_bwd(const sap_plan_t* p, const sap_slot_t* slots, int32_t rank, sap_code_t* codes, int32_t cap) {
  if (!p || !slots || rank < 0 || rank >= p->n_chunks || cap < 0 || (cap > 0 && !codes)) return -SAP_ERR_INVALID_ARG;
  const int32_t n_items = (int32_t)p->items.size();
  std::vector<sap_code_t> out;
  auto transfer = [&](int32_t stage, int32_t tensor, int32_t src, int32_t dst, int32_t x) {
    if (rank == src) out.push_back({stage, SAP_OP_SEND, tensor, dst, x});
    if (rank == dst) { out.push_back({stage, SAP_OP_RECV, tensor, src, x}); out.push_back({stage, SAP_OP_COPY, tensor, src, x}); }
  };
  for (int32_t x = 0; x < n_items; ++x) {
    const sap_item_t& im = p->items[x];
    const int32_t i = im.q_chunk, j = im.kv_chunk, R = slots[x].rank, st = slots[x].stage;
    if (R != i && R != j) return -SAP_ERR_INVALID_ARG;
    if (R == rank) out.push_back({st, SAP_OP_COMPUTING, -1, -1, x});
    if (i == j) continue;
    if (R == i) {  // K/V_j travels j -> i, the dK/dV contribution travels back
      transfer(st - 1, SAP_T_KV, j, i, x);
      transfer(st + 1, SAP_T_DKV, i, j, x);
    } else {       // Q_i and dO_i (with LSE, D) travel i -> j, the dQ contribution travels back
      transfer(st - 1, SAP_T_Q, i, j, x);
      transfer(st - 1, SAP_T_DO, i, j, x);
      transfer(st + 1, SAP_T_DQ, j, i, x);
    }
  }
  return emit_codes(out, codes, cap);
}

int32_t sap_debug_tile_program(const sap_plan_t* p, int32_t kind, int32_t a, int32_t b, int32_t* tiles, int32_t tiles_cap,
                               int32_t* segs, int32_t segs_cap, int32_t* n_segs) {
  if (!p || !n_segs || tiles_cap < 0 || segs_cap < 0) return -SAP_ERR_INVALID_ARG;
  TileProgram built;
  const TileProgram* prog = &built;
  const int32_t n_items = (int32_t)p->items.size();
  auto items_ok = [&]() { return a >= 0 && b >= a && b <= n_items; };
  auto chunks_ok = [&]() { return a >= 0 && b >= a && b <= p->n_chunks; };
  switch (kind) {
    case 0: prog = &p->fwd; break;
    case 1: prog = &p->kv; break;
    case 2: prog = &p->kv2; break;
    case 3: if (!items_ok()) return -SAP_ERR_INVALID_ARG; build_q_program(*p, a, b, built, false); break;
    case 4: if (!items_ok()) return -SAP_ERR_INVALID_ARG; build_q_program(*p, a, b, built, true); break;
    case 5: if (!chunks_ok()) return -SAP_ERR_INVALID_ARG; build_q_program(*p, p->chunk_offsets[a], p->chunk_offsets[b], built, true); break;
    case 6: case 7: if (!chunks_ok()) return -SAP_ERR_INVALID_ARG; build_kv_program(*p, built, a, b, kind == 7 ? 2 * kTile : kTile); break;
    case 10: prog = &p->fwd2; break;
    case 8: case 9: if (!items_ok()) return -SAP_ERR_INVALID_ARG; build_kv_program(*p, built, 0, -1, kind == 9 ? 2 * kTile : kTile, a, b, true); break;
    default: return -SAP_ERR_INVALID_ARG;
  }
  static_assert(sizeof(TileDesc) == 4 * sizeof(int32_t) && sizeof(SegDesc) == 8 * sizeof(int32_t), "flat int32 records");
  const int32_t nt = (int32_t)prog->tiles.size(), ns = (int32_t)prog->segs.size();
  *n_segs = ns;
  if (tiles && nt > 0 && nt <= tiles_cap) std::memcpy(tiles, prog->tiles.data(), sizeof(TileDesc) * nt);
  if (segs && ns > 0 && ns <= segs_cap) std::memcpy(segs, prog->segs.data(), sizeof(SegDesc) * ns);
  return nt;
}

const char* sap_strerror(int status) {
  switch (status) {
    case SAP_OK: return "ok";
    case SAP_ERR_INVALID_ARG: return "invalid argument";
    case SAP_ERR_BAD_CU_SEQLENS: return "bad cu_seqlens (must start at 0, be non-decreasing, end > 0)";
    case SAP_ERR_INDIVISIBLE: return "total length is not divisible by n_chunks";
    case SAP_ERR_UNSUPPORTED: return "unsupported configuration (head_dim in {64,128}, Hq % Hkv == 0, 16-byte aligned pointers)";
    case SAP_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
    case SAP_ERR_WRONG_ARCH: return "device is not sm_100 (B200)";
    case SAP_ERR_CUDA: return "CUDA error (see sap_last_cuda_error)";
    case SAP_ERR_NO_DEVICE: return "no CUDA device";
    case SAP_ERR_PLAN_MISMATCH: return "plan mismatch (n_tokens differs from the plan's, or the plan lives on another device)";
    case SAP_ERR_STATIC_LIMIT: return "problem too large for the built-in scratch memory of sap_attn_bwd_static (SAP_STATIC_WORKSPACE_BYTES)";
    default: return "unknown status";
  }
}

}  // extern "C"
