// Forward kernel: one CTA = one 128-row Q tile x one q-head, two CTAs per SM.
//
// Implements the `computing` instruction of PAPER.md Table 1 (:85-98) for every plan item the Q tile
// touches, with the "copy and rescale" merge (:239) fused: the running (max, sum, O) carried across a
// tile's items IS the exact log-sum-exp merge of the per-item partials (:59, Milakov & Gimelshein).
//
// Roles (256 threads):  warp 0 lane 0 = TMA producer;  warp 1 = tcgen05 issuer (+ TMEM alloc);
// warps 4-7 = softmax / correction / epilogue, one thread per Q row (TMEM lane = row, so row
// reductions need no shuffles).  Inside a CTA the chain S=QK^T -> softmax -> O+=PV is serial; the
// second resident CTA of the SM fills the tensor pipe while this one does softmax.
//
// TMEM (256 columns): [0,128) S fp32, overwritten in place by P bf16 in [0,64); [128,128+D) O fp32.
#pragma once
#include <cuda_bf16.h>
#include <math_constants.h>
#include "sap_internal.h"
#include "sm100_ptx.cuh"

namespace sap {

#ifdef SAP_TRACE  // instrumented build only (never the shipped library): SM cycle stamps of one CTA
__device__ unsigned long long g_sap_trace[128 * 64];
#define SAP_STAMP(iter, slot) do { if (blockIdx.x == 0 && (iter) < 128) g_sap_trace[(iter) * 64 + (slot)] = clock64(); } while (0)
// CTA pairs: slots [0,32) of the leader (block 0), [32,64) of its peer (block 1); the two SMs' clocks are not aligned
#define SAP_STAMP2(iter, slot) do { if (blockIdx.x < 2 && (iter) < 128) g_sap_trace[(iter) * 64 + 32 * blockIdx.x + (slot)] = clock64(); } while (0)
#define SAP_STAMP_MAX(iter, slot) do { if (blockIdx.x < 2 && (iter) < 128) atomicMax(&g_sap_trace[(iter) * 64 + 32 * blockIdx.x + (slot)], (unsigned long long)clock64()); } while (0)
#define SAP_STAMP_MIN(iter, slot) do { if (blockIdx.x < 2 && (iter) < 128) atomicMin(&g_sap_trace[(iter) * 64 + 32 * blockIdx.x + (slot)], (unsigned long long)clock64()); } while (0)
#else
#define SAP_STAMP(iter, slot) do { } while (0)
#define SAP_STAMP_MAX(iter, slot) do { } while (0)
#define SAP_STAMP_MIN(iter, slot) do { } while (0)
#define SAP_STAMP2(iter, slot) do { } while (0)
#endif

constexpr int kFwdThreads = 256;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kRescaleThreshold = 8.0f;  // log2 units: P stays <= 2^8, exact after final 1/l

template <int D>
struct FwdSmem {
  static constexpr int kTileBytes = kTile * D * 2;          // one Q / K / V tile
  static constexpr int kBoxBytes = kTile * 128;             // one TMA box: 128 rows x 128 B (64 bf16)
  static constexpr int kBoxes = D / 64;
  static constexpr int kBarOffset = 3 * kTileBytes;
  static constexpr int kTotal = 3 * kTileBytes + 128 + 1024;  // + barriers + alignment slack
};

// first document start <= t, i.e. cu[doc(t)]; cu has n_docs + 1 entries (PAPER.md:45 cu_len)
__device__ __forceinline__ int32_t doc_start_of(const int32_t* __restrict__ cu, int n_docs, int32_t t) {
  int lo = 0, hi = n_docs;  // invariant: cu[lo] <= t < cu[hi]
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(cu + mid) <= t) lo = mid; else hi = mid;
  }
  return __ldg(cu + lo);
}

// Grid order: kv-head-major, tiles longest-first inside a head.  The CTAs that run side by side then work on the same
// kv-head, whose K/V (and the Q / dO / dQ rows of its q-heads) fit in the 126 MB L2, instead of on all heads at once.
__device__ __forceinline__ void q_block_coords(int n_q_heads, int n_kv_heads, int& tile_idx, int& h) {
  const int g = n_q_heads / n_kv_heads, per_head = (gridDim.x / n_q_heads) * g;
  const int hk = blockIdx.x / per_head, rem = blockIdx.x % per_head;
  tile_idx = rem / g;
  h = hk * g + rem % g;
}
__device__ __forceinline__ void kv_block_coords(int n_kv_heads, int& tile_idx, int& hk) {
  const int n_tiles = gridDim.x / n_kv_heads;
  hk = blockIdx.x / n_tiles;
  tile_idx = blockIdx.x % n_tiles;
}

template <int D, bool PARTIAL>
__global__ void __launch_bounds__(kFwdThreads, 2)
sap_fwd_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapK,
               const __grid_constant__ CUtensorMap mapV, const TileDesc* __restrict__ tiles,
               const SegDesc* __restrict__ segs, const int32_t* __restrict__ cu, int n_docs,
               __nv_bfloat16* __restrict__ out, float* __restrict__ out_f32, float* __restrict__ lse,
               int n_tokens, int n_q_heads, int n_kv_heads, float scale_log2) {
  using L = FwdSmem<D>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t sQ = smem_u32(smem), sK = sQ + L::kTileBytes, sV = sK + L::kTileBytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::kBarOffset);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::kBarOffset + 96);
  const uint32_t bar_q_full = smem_u32(bars + 0), bar_k_full = smem_u32(bars + 1), bar_k_empty = smem_u32(bars + 2),
                 bar_v_full = smem_u32(bars + 3), bar_v_empty = smem_u32(bars + 4), bar_s_full = smem_u32(bars + 5),
                 bar_p_full = smem_u32(bars + 6) /* +1: second half of P */, bar_o_full = smem_u32(bars + 8);

  // logical warp id: the service warps (0-3: TMA, tcgen05 issuer, ...) are the physically LAST four warps, because the
  // SM's warp arbiter favours high warp ids and the single issuing threads must never starve; +4 keeps warp % 4
  // (the TMEM lane quarter) and the warpgroup split of setmaxnreg intact
  const int warp = ((threadIdx.x >> 5) + 4) & 7, lane = threadIdx.x & 31;
  int tile_idx, h;
  q_block_coords(n_q_heads, n_kv_heads, tile_idx, h);
  const int hk = h / (n_q_heads / n_kv_heads);
  const TileDesc td = tiles[tile_idx];

  if (threadIdx.x == 0) {
    mbar_init(bar_q_full, 1); mbar_init(bar_k_full, 1); mbar_init(bar_k_empty, 1);
    mbar_init(bar_v_full, 1); mbar_init(bar_v_empty, 1); mbar_init(bar_s_full, 1);
    mbar_init(bar_p_full, 128); mbar_init(bar_p_full + 8, 128); mbar_init(bar_o_full, 1);
    fence_mbar_init();
    tma_prefetch_desc(&mapQ); tma_prefetch_desc(&mapK); tma_prefetch_desc(&mapV);
  }
  if (warp == 1) { tmem_alloc(smem_u32(tmem_slot), 256); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t tS = tmem, tP = tmem, tO = tmem + 128;

  int n_iters = 0;
  for (int s = td.seg_begin; s < td.seg_end; ++s) n_iters += (segs[s].t_end - segs[s].t_begin + kTile - 1) / kTile;

  if (warp == 0) {
    // ------------------------------------------------------------------ TMA producer
    reg_dealloc<56>();
    if (n_iters > 0 && elect_one()) {
      mbar_expect_tx(bar_q_full, L::kTileBytes);
#pragma unroll
      for (int b = 0; b < L::kBoxes; ++b) tma_load_2d(sQ + b * L::kBoxBytes, &mapQ, h * D + b * 64, td.row0, bar_q_full);
      int it = 0;
      for (int s = td.seg_begin; s < td.seg_end; ++s) {
        const int c_begin = segs[s].t_begin, c_end = segs[s].t_end;
        for (int c0 = c_begin; c0 < c_end; c0 += kTile, ++it) {
          mbar_wait(bar_k_empty, (it & 1) ^ 1);
          mbar_expect_tx(bar_k_full, L::kTileBytes);
#pragma unroll
          for (int b = 0; b < L::kBoxes; ++b) tma_load_2d(sK + b * L::kBoxBytes, &mapK, hk * D + b * 64, c0, bar_k_full);
          mbar_wait(bar_v_empty, (it & 1) ^ 1);
          mbar_expect_tx(bar_v_full, L::kTileBytes);
#pragma unroll
          for (int b = 0; b < L::kBoxes; ++b) tma_load_2d(sV + b * L::kBoxBytes, &mapV, hk * D + b * 64, c0, bar_v_full);
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------ tcgen05 issuer
    reg_dealloc<56>();
    if (n_iters > 0) {
      constexpr uint32_t idesc_s = make_idesc_bf16(128, 128, 0, 0);  // S[128x128] = Q (K-major) x K^T (K-major)
      constexpr uint32_t idesc_o = make_idesc_bf16(128, D, 0, 1);    // O[128xD]  = P (TMEM)   x V (MN-major)
      mbar_wait(bar_q_full, 0);
      for (int it = 0; it < n_iters; ++it) {
        mbar_wait(bar_k_full, it & 1);
        tc_fence_after();
        if (elect_one()) {
#pragma unroll
          for (int k = 0; k < D / 16; ++k) {
            const uint32_t off = (k / 4) * L::kBoxBytes + (k % 4) * 32;
            umma_ss(tS, make_smem_desc(sQ + off, 16, 1024), make_smem_desc(sK + off, 16, 1024), idesc_s, k > 0);
          }
          umma_commit(bar_k_empty);
          umma_commit(bar_s_full);
        }
        __syncwarp();
        mbar_wait(bar_v_full, it & 1);
#pragma unroll
        for (int half = 0; half < 2; ++half) {  // PV starts as soon as the first 64 keys of P are in TMEM
          mbar_wait(bar_p_full + 8 * half, it & 1);
          tc_fence_after();
          if (elect_one()) {
#pragma unroll
            for (int k = half * 4; k < half * 4 + 4; ++k)  // 16 keys per MMA: 2 groups of 8 rows (SBO 1024 B); d blocks LBO apart
              umma_ts(tO, tP + k * 8, make_smem_desc(sV + k * 2048, L::kBoxBytes, 1024), idesc_o, (it > 0 || k > 0) ? 1u : 0u);
            if (half == 1) {
              umma_commit(bar_v_empty);
              if (it == n_iters - 1) umma_commit(bar_o_full);
            }
          }
          __syncwarp();
        }
        __syncwarp();
      }
    }
  } else if (warp < 4) {
    reg_dealloc<56>();
  } else {
    // ------------------------------------------------------------------ softmax / correction / epilogue
    reg_alloc<200>();
    const int r = (warp - 4) * 32 + lane;
    const int t = td.row0 + r;
    const bool valid = r < td.rows;
    const uint32_t lane_base = static_cast<uint32_t>((warp - 4) * 32) << 16;
    const int32_t doc_lo = valid ? doc_start_of(cu, n_docs, t) : 0;
    float m_used = -CUDART_INF_F;  // reference max (log2 domain) the running sum and O are scaled by
    float l_run = 0.f;
    int it = 0;
    for (int s = td.seg_begin; s < td.seg_end; ++s) {
      const SegDesc sd = segs[s];
      int lo = max(doc_lo, sd.kv_lo), hi = min(t + 1, sd.kv_hi);  // visible keys of this row: [lo, hi)
      if (!valid || t < sd.q_lo || t >= sd.q_hi) { lo = 0; hi = 0; }
      for (int c0 = sd.t_begin; c0 < sd.t_end; c0 += kTile, ++it) {
        mbar_wait(bar_s_full, it & 1);
        tc_fence_after();
        const bool need_mask = __any_sync(0xffffffffu, (c0 < lo) || (c0 + kTile > hi));
        // the whole S row of this thread: 128 fp32 in registers, one TMEM read
        uint32_t sv[128];
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
          if (it > 0) {
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
        // P = 2^(S*scale_log2 - m) (masked entries: 2^-inf = 0), row sum, bf16 P back into TMEM over S
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
          mbar_arrive(bar_p_full + 8 * half);
        }
        {
          float a0, a1;
          unpack_f32x2(add_f32x2(add_f32x2(ls2[0], ls2[1]), add_f32x2(ls2[2], ls2[3])), a0, a1);
          l_run += a0 + a1;
        }
      }
    }
    // ---- epilogue: O / l -> global, LSE (natural log, PAPER.md silent: SURVEY A-11)
    if (n_iters > 0) {
      mbar_wait(bar_o_full, 0);
      tc_fence_after();
    }
    const float inv_l = l_run > 0.f ? 1.f / l_run : 0.f;
    const size_t row_off = (static_cast<size_t>(t) * n_q_heads + h) * D;
#pragma unroll
    for (int c = 0; c < D / 32; ++c) {
      uint32_t v[32];
      if (n_iters > 0) {
        tmem_ld32(tO + lane_base + c * 32, v);
        tmem_wait_ld();
      } else {
#pragma unroll
        for (int i = 0; i < 32; ++i) v[i] = 0u;
      }
      if (valid) {
        if (PARTIAL) {
          float4* dst = reinterpret_cast<float4*>(out_f32 + row_off + c * 32);
#pragma unroll
          for (int i = 0; i < 8; ++i)
            dst[i] = make_float4(__uint_as_float(v[4 * i]) * inv_l, __uint_as_float(v[4 * i + 1]) * inv_l,
                                 __uint_as_float(v[4 * i + 2]) * inv_l, __uint_as_float(v[4 * i + 3]) * inv_l);
        } else {
          uint4* dst = reinterpret_cast<uint4*>(out + row_off + c * 32);
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            uint4 w;
            w.x = pack_bf16x2(__uint_as_float(v[8 * i + 0]) * inv_l, __uint_as_float(v[8 * i + 1]) * inv_l);
            w.y = pack_bf16x2(__uint_as_float(v[8 * i + 2]) * inv_l, __uint_as_float(v[8 * i + 3]) * inv_l);
            w.z = pack_bf16x2(__uint_as_float(v[8 * i + 4]) * inv_l, __uint_as_float(v[8 * i + 5]) * inv_l);
            w.w = pack_bf16x2(__uint_as_float(v[8 * i + 6]) * inv_l, __uint_as_float(v[8 * i + 7]) * inv_l);
            dst[i] = w;
          }
        }
      }
    }
    if (valid)
      lse[static_cast<size_t>(h) * n_tokens + t] = l_run > 0.f ? (m_used + log2f(l_run)) * kLn2 : -CUDART_INF_F;
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, 256);
}

}  // namespace sap
