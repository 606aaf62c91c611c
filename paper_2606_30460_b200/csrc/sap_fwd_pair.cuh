// Forward kernel, pair form: one work item = one 128-row Q tile x TWO q-heads of one GQA group; PERSISTENT: one CTA per
// SM takes work items off a global counter in the launch order (kv-head-major, longest tile first), so barriers, TMEM
// and the K/V ring are set up once and the next item's Q / first K/V loads and first S run under the current item's tail.
// (`computing` of PAPER.md Table 1 (:85-98) with the "copy and rescale" merge (:239) fused, as in sap_fwd.cuh.)
//
// The two heads attend the same rows to the same keys, so they walk the same segments and share every K / V tile
// in shared memory (one TMA fill per two score tiles).  Two softmax warpgroups (A, B: one thread per row) alternate
// on the MUFU pipe while the tensor pipe runs the other head's GEMMs:
//     tensor pipe:  ... PV_A(i)  S_A(i+1)  PV_B(i)  S_B(i+1)  PV_A(i+1) ...
//     warpgroup A:      softmax_A(i+1) ----------------->
//     warpgroup B:                          softmax_B(i+1) ----------------->
// Used when Hq/Hkv is even; sap_fwd_kernel (one head per CTA, two CTAs per SM) serves the other shapes.
//
// Roles (384 threads): warpgroups A and B = softmax / correction / epilogue; service warpgroup = TMA producer
// (one elected thread) and tcgen05 issuer (one elected thread).
// TMEM (512 columns): [0,128) S_A -> P_A | [128,256) S_B -> P_B | [256,256+D) O_A | [384,384+D) O_B.
#pragma once
#include "sap_fwd.cuh"

namespace sap {

#define FWD_STAMP(iter, slot) SAP_STAMP(iter, slot)

constexpr int kFwdPairThreads = 384;
constexpr int kFwdPairStages = 2;  // K and V rings

template <int D>
struct FwdPairSmem {
  static constexpr int kTileBytes = kTile * D * 2;
  static constexpr int kBoxBytes = kTile * 128;
  static constexpr int kBoxes = D / 64;
  static constexpr int kOffQ = 0;                                   // Q_A, Q_B
  static constexpr int kOffK = 2 * kTileBytes;                      // K ring
  static constexpr int kOffV = kOffK + kFwdPairStages * kTileBytes; // V ring
  static constexpr int kBarOffset = kOffV + kFwdPairStages * kTileBytes;
  static constexpr int kTotal = kBarOffset + 512;   // barriers [0,192) | TMEM slot 200 | work ring [256, 256 + 2 x 96)
};

// Work item w of a launch -> (kv-head, Q tile, first q-head of the pair): kv-head-major, tiles longest-first inside a
// head, the g/2 head pairs of a tile adjacent (CTAs that run side by side share one kv-head's K/V in L2).
// Two forms of a work item's two 128-row units: head pairs (row_pair = 0: units A, B = q-heads h0, h0 + 1 of one GQA group on
// the same 128 rows; even Hq/Hkv) and row pairs (row_pair = 1: rows [row0, +128) and [row0 + 128, +128) of ONE q-head, over
// a 256-row tile program; any Hq/Hkv, used for the odd ones, e.g. MHA).  Either way both units stream the same K/V tiles.
struct FwdPairWork { int hk, tile_idx, h0; };
__device__ __forceinline__ FwdPairWork fwd_pair_work(int w, int n_tiles, int g, int row_pair) {
  const int pairs = row_pair ? g : g / 2, per_head = n_tiles * pairs;
  const int hk = w / per_head, rem = w % per_head;
  return {hk, rem / pairs, hk * g + (row_pair ? 1 : 2) * (rem % pairs)};
}
// One slot of the work ring the scheduler thread fills ahead of the other roles: everything they need to start an item
// without a global load of their own (tile, first segment, iteration count, and the cu_seqlens entries around the tile's
// first row, from which each row finds the start of its document).
constexpr int kFwdCuWindow = 8;
struct FwdWorkSlot {
  int32_t w;            // work item, -1 = no more work
  int32_t row0, rows, seg_begin, seg_end;
  int32_t n_iters;      // streamed K/V tiles of the item
  int32_t n_cu;         // valid entries of cu_win
  int32_t pad;
  int32_t cu_win[kFwdCuWindow];   // cu[e0 .. e0 + n_cu), e0 = document of row0
  SegDesc seg0;         // segs[seg_begin] (valid if n_iters > 0)
};
static_assert(sizeof(FwdWorkSlot) == 96, "work ring slot layout");

__device__ __forceinline__ int fwd_tile_iters(const TileDesc& td, const SegDesc* __restrict__ segs) {
  int n = 0;
  for (int s = td.seg_begin; s < td.seg_end; ++s) n += (segs[s].t_end - segs[s].t_begin + kTile - 1) / kTile;
  return n;
}

// `sched` = {next, done}: two zero-initialised counters of this launch.  CTA b starts with item b and then takes item
// gridDim.x + atomicAdd(next, 1); the last CTA to leave zeroes both again, so the pair can serve the next launch.
// The host hands every launch a pair no other launch in flight holds (sap_api.cu: next_sched_pair).
template <int D, bool PARTIAL>
__global__ void __launch_bounds__(kFwdPairThreads, 1)
sap_fwd_pair_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapK,
                    const __grid_constant__ CUtensorMap mapV, const TileDesc* __restrict__ tiles,
                    const SegDesc* __restrict__ segs, const int32_t* __restrict__ cu, int n_docs,
                    __nv_bfloat16* __restrict__ out, float* __restrict__ out_f32, float* __restrict__ lse,
                    int n_tokens, int n_q_heads, int n_kv_heads, float scale_log2, int n_tiles, int n_work,
                    int* __restrict__ sched, int row_pair) {
  using L = FwdPairSmem<D>;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = smem_raw;
  if (smem_u32(smem) & 1023u) __trap();
  const uint32_t s0 = smem_u32(smem);
  const uint32_t sQ = s0 + L::kOffQ, sK = s0 + L::kOffK, sV = s0 + L::kOffV;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::kBarOffset);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::kBarOffset + 200);
  volatile FwdWorkSlot* work_ring = reinterpret_cast<volatile FwdWorkSlot*>(smem + L::kBarOffset + 256);   // 2 slots
  const uint32_t bar_q_full = smem_u32(bars + 0), bar_k_full = smem_u32(bars + 1), bar_k_empty = smem_u32(bars + 3),
                 bar_v_full = smem_u32(bars + 5), bar_v_empty = smem_u32(bars + 7),
                 bar_s_full = smem_u32(bars + 9) /* [A, B] */, bar_p_full = smem_u32(bars + 11) /* [A0, A1, B0, B1] */,
                 bar_o_full = smem_u32(bars + 15) /* [A, B] */, bar_q_empty = smem_u32(bars + 17),
                 bar_o_empty = smem_u32(bars + 18) /* [A, B] */, bar_w_full = smem_u32(bars + 20) /* [2] */,
                 bar_w_empty = smem_u32(bars + 22) /* [2] */;

  // logical warp id: the service warpgroup (logical warps 0-3) is the physically last one (see sap_fwd.cuh)
  const int warp = ((threadIdx.x >> 5) + 4) % (kFwdPairThreads / 32), lane = threadIdx.x & 31;
  const int g = n_q_heads / n_kv_heads;

  if (threadIdx.x == 0) {
    mbar_init(bar_q_full, 1); mbar_init(bar_q_empty, 1);
    for (int i = 0; i < kFwdPairStages; ++i) {
      mbar_init(bar_k_full + 8 * i, 1); mbar_init(bar_k_empty + 8 * i, 1);
      mbar_init(bar_v_full + 8 * i, 1); mbar_init(bar_v_empty + 8 * i, 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(bar_s_full + 8 * i, 1); mbar_init(bar_o_full + 8 * i, 1); mbar_init(bar_o_empty + 8 * i, 4);
      mbar_init(bar_w_full + 8 * i, 1); mbar_init(bar_w_empty + 8 * i, 1 + 8);   // issuer + 8 softmax warps
    }
    for (int i = 0; i < 4; ++i) mbar_init(bar_p_full + 8 * i, 4);   // one arrival per softmax warp
    fence_mbar_init();
    tma_prefetch_desc(&mapQ); tma_prefetch_desc(&mapK); tma_prefetch_desc(&mapV);
  }
  if (warp == 1) { tmem_alloc(smem_u32(tmem_slot), 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  if (warp < 4) {
    reg_dealloc<88>();
    if (warp == 0) {
      // ---------------------------------------------------------------- scheduler + TMA producer
      if (elect_one()) {
        int st = 0, ph = 1;  // K/V rings run on across work items; empty barriers: the first pass must not block
        int ws = 0, wph = 1, nq = 0;   // work ring slot / phase; items with loads so far
        for (int w = blockIdx.x;; w = gridDim.x + atomicAdd(sched, 1)) {
          const bool end = w >= n_work;
          FwdPairWork wk = {0, 0, 0};
          TileDesc td = {0, 0, 0, 0};
          int n_it = 0, e0 = 0, n_cu = 0;
          if (!end) {   // all global loads of the item's metadata happen here, ahead of the roles that use it
            wk = fwd_pair_work(w, n_tiles, g, row_pair);
            td = tiles[wk.tile_idx];
            n_it = fwd_tile_iters(td, segs);
            int lo = 0, hi = n_docs;   // e0 = document of row0: cu[e0] <= row0 < cu[hi]
            while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(cu + mid) <= td.row0) lo = mid; else hi = mid; }
            e0 = lo;
            n_cu = min(kFwdCuWindow, n_docs + 1 - e0);
          }
          mbar_wait(bar_w_empty + 8 * ws, wph);
          volatile FwdWorkSlot* slot = work_ring + ws;
          slot->w = end ? -1 : w;
          if (!end) {
            slot->row0 = td.row0; slot->rows = td.rows; slot->seg_begin = td.seg_begin; slot->seg_end = td.seg_end;
            slot->n_iters = n_it; slot->n_cu = n_cu;
            for (int j = 0; j < n_cu; ++j) slot->cu_win[j] = __ldg(cu + e0 + j);
            if (n_it > 0) {
              const SegDesc sd = segs[td.seg_begin];
              slot->seg0.t_begin = sd.t_begin; slot->seg0.t_end = sd.t_end; slot->seg0.q_lo = sd.q_lo; slot->seg0.q_hi = sd.q_hi;
              slot->seg0.kv_lo = sd.kv_lo; slot->seg0.kv_hi = sd.kv_hi; slot->seg0.item = sd.item;
            }
          }
          mbar_arrive(bar_w_full + 8 * ws);   // release: the slot is written
          if (++ws == 2) { ws = 0; wph ^= 1; }
          if (end) break;
          if (n_it == 0) continue;
          mbar_wait(bar_q_empty, (nq & 1) ^ 1);   // the last S of the previous item has read Q
          ++nq;
          mbar_expect_tx(bar_q_full, 2 * L::kTileBytes);
#pragma unroll
          for (int x = 0; x < 2; ++x)
#pragma unroll
            for (int b = 0; b < L::kBoxes; ++b)
              tma_load_2d(sQ + x * L::kTileBytes + b * L::kBoxBytes, &mapQ, (wk.h0 + (row_pair ? 0 : x)) * D + b * 64,
                          td.row0 + (row_pair ? kTile * x : 0), bar_q_full);   // rows past the end of the tensor are zero-filled
          for (int s = td.seg_begin; s < td.seg_end; ++s) {
            const int c_begin = segs[s].t_begin, c_end = segs[s].t_end;
            for (int c0 = c_begin; c0 < c_end; c0 += kTile) {
              mbar_wait(bar_k_empty + 8 * st, ph);
              mbar_expect_tx(bar_k_full + 8 * st, L::kTileBytes);
#pragma unroll
              for (int b = 0; b < L::kBoxes; ++b)
                tma_load_2d(sK + st * L::kTileBytes + b * L::kBoxBytes, &mapK, wk.hk * D + b * 64, c0, bar_k_full + 8 * st);
              mbar_wait(bar_v_empty + 8 * st, ph);
              mbar_expect_tx(bar_v_full + 8 * st, L::kTileBytes);
#pragma unroll
              for (int b = 0; b < L::kBoxes; ++b)
                tma_load_2d(sV + st * L::kTileBytes + b * L::kBoxBytes, &mapV, wk.hk * D + b * 64, c0, bar_v_full + 8 * st);
              if (++st == kFwdPairStages) { st = 0; ph ^= 1; }
            }
          }
        }
      }
    } else if (warp == 1) {
      // ---------------------------------------------------------------- tcgen05 issuer (one elected thread)
      if (elect_one()) {
        constexpr uint32_t idesc_s = make_idesc_bf16(128, 128, 0, 0);  // S[128x128] = Q (K-major) x K^T (K-major)
        constexpr uint32_t idesc_o = make_idesc_bf16(128, D, 0, 1);    // O[128xD]  = P (TMEM)   x V (MN-major)
        auto issue_s = [&](int x, int st) {   // S_x = Q_x K^T for the K tile in stage st
#pragma unroll
          for (int k = 0; k < D / 16; ++k) {
            const uint32_t off = (k / 4) * L::kBoxBytes + (k % 4) * 32;
            umma_ss(tmem + 128 * x, make_smem_desc(sQ + x * L::kTileBytes + off, 16, 1024),
                    make_smem_desc(sK + st * L::kTileBytes + off, 16, 1024), idesc_s, k > 0);
          }
          umma_commit(bar_s_full + 8 * x);
        };
        int st = 0, ph = 0;   // stage / phase of the current iteration; run on across work items
        int gi = 0;           // iterations so far (parity of the P barriers)
        int nq = 0;           // items with work so far (parity of the Q / O barriers)
        int ws = 0, wph = 0;
        for (;;) {
          mbar_wait(bar_w_full + 8 * ws, wph);
          const int w = work_ring[ws].w, n_iters = work_ring[ws].n_iters;
          mbar_arrive(bar_w_empty + 8 * ws);
          if (++ws == 2) { ws = 0; wph ^= 1; }
          if (w < 0) break;
          if (n_iters == 0) continue;
          auto issue_pv = [&](int x, int st_, int it) {  // O_x += P_x V, in two halves of 64 keys
#pragma unroll
            for (int half = 0; half < 2; ++half) {
              mbar_wait(bar_p_full + 8 * (2 * x + half), gi & 1);
              tc_fence_after();
#pragma unroll
              for (int k = half * 4; k < half * 4 + 4; ++k)  // 16 keys per MMA: 2 groups of 8 rows (SBO 1024 B)
                umma_ts(tmem + 256 + 128 * x, tmem + 128 * x + k * 8,
                        make_smem_desc(sV + st_ * L::kTileBytes + k * 2048, L::kBoxBytes, 1024), idesc_o,
                        (it > 0 || k > 0) ? 1u : 0u);
            }
            if (it == n_iters - 1) umma_commit(bar_o_full + 8 * x);
          };
          mbar_wait(bar_q_full, nq & 1);
          mbar_wait(bar_k_full + 8 * st, ph);
          tc_fence_after();
          issue_s(0, st);
          issue_s(1, st);
          umma_commit(bar_k_empty + 8 * st);
          if (n_iters == 1) umma_commit(bar_q_empty);   // the item's last S has been issued: Q may be overwritten once it is done
          if (nq > 0) {   // the previous item's O_A, O_B have left TMEM (long before the first P of this item is ready)
            mbar_wait(bar_o_empty, (nq - 1) & 1);
            mbar_wait(bar_o_empty + 8, (nq - 1) & 1);
            tc_fence_after();
          }
          for (int it = 0; it < n_iters; ++it, ++gi) {
            const int st_n = (st + 1 == kFwdPairStages) ? 0 : st + 1, ph_n = (st_n == 0) ? ph ^ 1 : ph;
            const bool more = it + 1 < n_iters;
            FWD_STAMP(it, 0);
            mbar_wait(bar_v_full + 8 * st, ph);
            FWD_STAMP(it, 1);
            issue_pv(0, st, it);
            FWD_STAMP(it, 2);
            if (more) {
              mbar_wait(bar_k_full + 8 * st_n, ph_n);
              tc_fence_after();
              issue_s(0, st_n);   // S_A(it+1) runs while warpgroup B is still in softmax_B(it)
            }
            FWD_STAMP(it, 3);
            issue_pv(1, st, it);
            FWD_STAMP(it, 4);
            umma_commit(bar_v_empty + 8 * st);
            if (more) {
              issue_s(1, st_n);
              umma_commit(bar_k_empty + 8 * st_n);
              if (it + 2 == n_iters) umma_commit(bar_q_empty);
            }
            st = st_n; ph = ph_n;
          }
          ++nq;
        }
      }
    }
  } else {
    // ------------------------------------------------------------------ softmax / correction / epilogue (A or B)
    reg_alloc<208>();  // 256 x 208 + 128 x 88 = the 384 x 168 register pool
    const int x = (warp - 4) >> 2;  // 0: head h0 (A), 1: head h0 + 1 (B)
    const int r = (warp & 3) * 32 + lane;
    const uint32_t lane_base = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t tS = tmem + 128 * x, tP = tS, tO = tmem + 256 + 128 * x;
    const uint32_t bar_s = bar_s_full + 8 * x, bar_p = bar_p_full + 16 * x, bar_o = bar_o_full + 8 * x,
                   bar_oe = bar_o_empty + 8 * x;
    int gi = 0, nq = 0, ws = 0, wph = 0;
    for (;;) {
      mbar_wait(bar_w_full + 8 * ws, wph);
      volatile FwdWorkSlot* slot = work_ring + ws;
      const int w = slot->w;
      TileDesc td = {0, 0, 0, 0};
      SegDesc sd = {0, 0, 0, 0, 0, 0, 0, 0};
      int n_iters = 0, t = 0;
      int32_t doc_lo = 0;
      bool valid = false, far = false;
      if (w >= 0) {
        td.row0 = slot->row0; td.rows = slot->rows; td.seg_begin = slot->seg_begin; td.seg_end = slot->seg_end;
        n_iters = slot->n_iters;
        const int r_unit = (row_pair ? kTile * x : 0) + r;   // row inside the tile (row pairs: unit B = rows 128..255)
        t = td.row0 + r_unit;
        valid = r_unit < td.rows;
        const int n_cu = slot->n_cu;
        doc_lo = slot->cu_win[0];   // start of the row's document: the last window entry <= t (cu is non-decreasing)
#pragma unroll
        for (int j = 1; j < kFwdCuWindow; ++j) {
          const int32_t c = slot->cu_win[j];
          if (j < n_cu && c <= t) doc_lo = c;
        }
        far = valid && n_cu == kFwdCuWindow && slot->cu_win[kFwdCuWindow - 1] <= t;   // more than 7 documents start inside the tile before this row
        if (n_iters > 0) {
          sd.t_begin = slot->seg0.t_begin; sd.t_end = slot->seg0.t_end; sd.q_lo = slot->seg0.q_lo; sd.q_hi = slot->seg0.q_hi;
          sd.kv_lo = slot->seg0.kv_lo; sd.kv_hi = slot->seg0.kv_hi;
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_w_empty + 8 * ws);
      if (++ws == 2) { ws = 0; wph ^= 1; }
      if (w < 0) break;
      if (far) doc_lo = doc_start_of(cu, n_docs, t);
      const FwdPairWork wk = fwd_pair_work(w, n_tiles, g, row_pair);
      const int h = wk.h0 + (row_pair ? 0 : x);
      float m_used = -CUDART_INF_F;  // reference max (log2 domain) the running sum and O are scaled by
      float l_run = 0.f;
      int it = 0;
      for (int s = td.seg_begin; s < td.seg_end; ++s) {
        // the next segment's descriptor is loaded one segment ahead (its latency hides behind this segment's tiles)
        const SegDesc sd_next = segs[s + 1 < td.seg_end ? s + 1 : s];
        int lo = max(doc_lo, sd.kv_lo), hi = min(t + 1, sd.kv_hi);  // visible keys of this row: [lo, hi)
        if (!valid || t < sd.q_lo || t >= sd.q_hi) { lo = 0; hi = 0; }
        const int c_end = sd.t_end;
        for (int c0 = sd.t_begin; c0 < c_end; c0 += kTile, ++it, ++gi) {
          mbar_wait(bar_s, gi & 1);
          tc_fence_after();
          if ((warp & 3) == 0 && lane == 0) FWD_STAMP(it, 16 + 8 * x);
          const bool need_mask = __any_sync(0xffffffffu, (c0 < lo) || (c0 + kTile > hi));
          uint32_t sv[128];  // the whole S row of this thread
#pragma unroll
          for (int c = 0; c < 4; ++c) tmem_ld32(tS + lane_base + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&sv[c * 32]));
          tmem_wait_ld();
          if (need_mask) {  // boundary tiles only (document start, diagonal, item edge)
#pragma unroll
            for (int i = 0; i < 128; ++i) {
              const int col = c0 + i;
              if (!(col >= lo && col < hi)) sv[i] = 0xff800000u;  // -inf
            }
          }
          float mx4[4] = {-CUDART_INF_F, -CUDART_INF_F, -CUDART_INF_F, -CUDART_INF_F};
#pragma unroll
          for (int i = 0; i < 128; i += 4) {
#pragma unroll
            for (int e = 0; e < 4; ++e) mx4[e] = fmaxf(mx4[e], __uint_as_float(sv[i + e]));
          }
          const float m_new = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * scale_log2;
          // lazy rescale: only when the max moved by more than 2^8 (or the row saw its first key)
          const bool grow = m_new > m_used + kRescaleThreshold || (m_used == -CUDART_INF_F && m_new > -CUDART_INF_F);
          if (__any_sync(0xffffffffu, grow)) {
            const float f = grow ? ((m_used == -CUDART_INF_F) ? 0.f : ex2_approx(m_used - m_new)) : 1.f;
            if (grow) { m_used = m_new; l_run *= f; }
            if (it > 0) {  // S(it) complete => PV(it-1) complete (tensor pipe order): O may be rewritten
#pragma unroll
              for (int c = 0; c < D / 32; ++c) {
                uint32_t v[32];
                tmem_ld32(tO + lane_base + c * 32, v);
                tmem_wait_ld();
#pragma unroll
                for (int i = 0; i < 32; ++i) v[i] = __float_as_uint(__uint_as_float(v[i]) * f);
                tmem_st32(tO + lane_base + c * 32, v);
              }
            }
          }
          const float neg_m = (m_used == -CUDART_INF_F) ? 0.f : -m_used;
          // packed fp32 pairs (FFMA2 / FADD2): the two softmax warps of a scheduler are issue-bound, not MUFU-bound
          const uint64_t sc2 = pack_f32x2(scale_log2, scale_log2), nm2 = pack_f32x2(neg_m, neg_m);
          uint64_t ls2[4] = {0ull, 0ull, 0ull, 0ull};   // four pairs of partial row sums
#pragma unroll
          for (int half = 0; half < 2; ++half) {
#pragma unroll
            for (int c = half * 2; c < half * 2 + 2; ++c) {
              uint32_t pk[16];
#pragma unroll
              for (int i = 0; i < 32; i += 2) {
                float x0, x1;
                unpack_f32x2(fma_f32x2(pack_f32x2(__uint_as_float(sv[c * 32 + i]), __uint_as_float(sv[c * 32 + i + 1])), sc2, nm2), x0, x1);
                const float p0 = ex2_approx(x0), p1 = ex2_approx(x1);
                ls2[(i >> 1) & 3] = add_f32x2(ls2[(i >> 1) & 3], pack_f32x2(p0, p1));
                pk[i >> 1] = pack_bf16x2(p0, p1);
              }
              tmem_st16(tP + lane_base + c * 16, pk);
            }
            tmem_wait_st();
            tc_fence_before();
            mbar_arrive_warp(bar_p + 8 * half);
            if ((warp & 3) == 0 && lane == 0) FWD_STAMP(it, 17 + 8 * x + half);
          }
          {
            float a0, a1;
            unpack_f32x2(add_f32x2(add_f32x2(ls2[0], ls2[1]), add_f32x2(ls2[2], ls2[3])), a0, a1);
            l_run += a0 + a1;
          }
        }
        sd = sd_next;
      }
      // ---- epilogue: O / l -> global, LSE (natural log).  O leaves TMEM first and the columns are handed back, so the
      // next item's first PV does not wait for the global stores.
      const float inv_l = l_run > 0.f ? 1.f / l_run : 0.f;
      const size_t row_off = (static_cast<size_t>(t) * n_q_heads + h) * D;
      uint32_t o[D];
      if (n_iters > 0) {
        mbar_wait(bar_o, nq & 1);
        tc_fence_after();
#pragma unroll
        for (int c = 0; c < D / 32; ++c) tmem_ld32(tO + lane_base + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&o[c * 32]));
        tmem_wait_ld();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_oe);
        ++nq;
      } else {
#pragma unroll
        for (int i = 0; i < D; ++i) o[i] = 0u;
      }
      if (valid) {
        if (PARTIAL) {
          float4* dst = reinterpret_cast<float4*>(out_f32 + row_off);
#pragma unroll
          for (int i = 0; i < D / 4; ++i)
            dst[i] = make_float4(__uint_as_float(o[4 * i]) * inv_l, __uint_as_float(o[4 * i + 1]) * inv_l,
                                 __uint_as_float(o[4 * i + 2]) * inv_l, __uint_as_float(o[4 * i + 3]) * inv_l);
        } else {
          uint4* dst = reinterpret_cast<uint4*>(out + row_off);
#pragma unroll
          for (int i = 0; i < D / 8; ++i) {
            uint4 wv;
            wv.x = pack_bf16x2(__uint_as_float(o[8 * i + 0]) * inv_l, __uint_as_float(o[8 * i + 1]) * inv_l);
            wv.y = pack_bf16x2(__uint_as_float(o[8 * i + 2]) * inv_l, __uint_as_float(o[8 * i + 3]) * inv_l);
            wv.z = pack_bf16x2(__uint_as_float(o[8 * i + 4]) * inv_l, __uint_as_float(o[8 * i + 5]) * inv_l);
            wv.w = pack_bf16x2(__uint_as_float(o[8 * i + 6]) * inv_l, __uint_as_float(o[8 * i + 7]) * inv_l);
            dst[i] = wv;
          }
        }
        lse[static_cast<size_t>(h) * n_tokens + t] = l_run > 0.f ? (m_used + log2f(l_run)) * kLn2 : -CUDART_INF_F;
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, 512);
  if (threadIdx.x == 0) {   // the last CTA to leave re-arms the counters for the next launch
    __threadfence();
    const int left = atomicAdd(sched + 1, 1);
    // A pair serves ONE launch at a time (sap.h, sap_attn_fwd).  Every CTA draws from `next` until its draw misses, so a
    // launch that had the pair to itself ends with done < gridDim.x and next == n_work; anything else means a second
    // launch was drawing from the same pair and work items were skipped or done twice: stop loudly, not with wrong output.
    if (left >= static_cast<int>(gridDim.x)) __trap();
    if (left == static_cast<int>(gridDim.x) - 1) {
      if (*reinterpret_cast<volatile int*>(sched) != n_work) __trap();
      sched[0] = 0; sched[1] = 0; __threadfence();
    }
  }
}

}  // namespace sap
