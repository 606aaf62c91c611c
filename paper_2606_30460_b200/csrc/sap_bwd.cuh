// Backward kernels (Table 1 tensors do / dq / dkv; fwd+bwd is what the paper times, :173).
//
//   sap_bwd_pre_kernel : D[h,t] = sum_c dO[t,h,c] * O[t,h,c]                 (HBM-bound)
//   sap_bwd_dq_kernel  : Q-stationary, walks the same tile program as the forward:
//                        S = QK^T, dP = dO V^T, dS = P*(dP - D), dQ += dS K   -> dQ bf16 directly
//   sap_bwd_dkv_kernel : KV-stationary, walks the transposed (per-kv-chunk) program, loops over the
//                        Hq/Hkv q-heads of the group: S^T = K Q^T, dP^T = V dO^T, dV += P^T dO, dK += dS^T Q
//
// With P = exp(scale*S - LSE) on the visible pairs.  No atomics, no fp32 dQ workspace, deterministic.
#pragma once
#include <cuda_bf16.h>
#include <math_constants.h>
#include "sap_fwd.cuh"
#include "sap_internal.h"
#include "sm100_ptx.cuh"

namespace sap {

// ------------------------------------------------------------------------------------------------
// D = rowsum(dO * O): one 16-lane (d=128) or 8-lane (d=64) group per (token, head), 16-byte loads,
// shuffle reduction inside the group.  Output fp32 [Hq, N].
// ------------------------------------------------------------------------------------------------
constexpr int kPreThreads = 256;

template <int D>
__global__ void __launch_bounds__(kPreThreads)
sap_bwd_pre_kernel(const __nv_bfloat16* __restrict__ dout, const __nv_bfloat16* __restrict__ out,
                   float* __restrict__ dsum, int64_t n_tokens, int n_q_heads, int64_t token_begin, int64_t token_count) {
  constexpr int G = D / 8;  // lanes per row, 8 bf16 each
  dout += token_begin * n_q_heads * D;   // tokens [token_begin, token_begin + token_count) only
  out += token_begin * n_q_heads * D;
  const int64_t n_rows = token_count * n_q_heads;
  const int64_t gthread = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
  const int64_t groups_total = static_cast<int64_t>(gridDim.x) * blockDim.x / G;
  const int gl = static_cast<int>(gthread % G);
  const int64_t n_rows_pad = (n_rows + groups_total - 1) / groups_total * groups_total;
  for (int64_t row = gthread / G; row < n_rows_pad; row += groups_total) {
    float acc = 0.f;
    if (row < n_rows) {
      const uint4 a = *reinterpret_cast<const uint4*>(dout + row * D + gl * 8);
      const uint4 b = *reinterpret_cast<const uint4*>(out + row * D + gl * 8);
      const uint32_t aw[4] = {a.x, a.y, a.z, a.w}, bw[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        acc = fmaf(__uint_as_float(aw[i] << 16), __uint_as_float(bw[i] << 16), acc);
        acc = fmaf(__uint_as_float(aw[i] & 0xffff0000u), __uint_as_float(bw[i] & 0xffff0000u), acc);
      }
    }
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (row < n_rows && gl == 0) {
      const int64_t t = token_begin + row / n_q_heads;
      const int h = static_cast<int>(row % n_q_heads);
      dsum[h * n_tokens + t] = acc;
    }
  }
}

// last document end > s, i.e. cu[doc(s) + 1]
__device__ __forceinline__ int32_t doc_end_of(const int32_t* __restrict__ cu, int n_docs, int32_t s) {
  int lo = 0, hi = n_docs;  // invariant: cu[lo] <= s < cu[hi]
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(cu + mid) <= s) lo = mid; else hi = mid;
  }
  return __ldg(cu + hi);
}

constexpr int kBwdN = 64;  // streamed tile rows in both backward kernels


// ------------------------------------------------------------------------------------------------
// dK/dV kernel.  One CTA = one 128-row K/V tile x one kv-head, one CTA per SM, 384 threads:
//   warp 0 TMA producer, warp 1 tcgen05 issuer, warp 2 LSE/D loader, warps 4-11 compute
//   (warp w: TMEM lane quarter w%4 = key rows, column half (w-4)/4 of the 64 streamed q rows).
// TMEM (512 columns): [0,128) dK, [128,256) dV, two score buffers b at 256+128b: S^T fp32 [0,64) with
//   P^T bf16 written over columns [32h, 32h+16) by the warp of half h; dP^T fp32 [64,128), dS^T likewise.
// The issuer runs one iteration ahead: S^T/dP^T of tile i+1 are in flight while tile i is in softmax.
// ------------------------------------------------------------------------------------------------
constexpr int kDkvParts = 4;                        // column parts of the 64 streamed q rows, one compute warp each
constexpr int kDkvThreads = 128 + 128 * kDkvParts;  // 4 service warps + 4 * kDkvParts compute warps
constexpr int kDkvCols = kBwdN / kDkvParts;        // q rows (TMEM columns) per compute warp
constexpr int kDkvStages = 3;

template <int D>
struct DkvSmem {
  static constexpr int kKVBytes = kTile * D * 2;   // K or V, 128 rows
  static constexpr int kQBytes = kBwdN * D * 2;    // Q or dO stage, 64 rows
  static constexpr int kKVBox = kTile * 128;
  static constexpr int kQBox = kBwdN * 128;
  static constexpr int kBoxes = D / 64;
  static constexpr int kOffK = 0, kOffV = kKVBytes, kOffQ = 2 * kKVBytes, kOffDO = 2 * kKVBytes + kDkvStages * kQBytes;
  static constexpr int kOffStat = kOffDO + kDkvStages * kQBytes;   // [stage][2][64] floats
  static constexpr int kBarOffset = kOffStat + kDkvStages * 512;
  static constexpr int kTotal = kBarOffset + 256;
};

template <int D>
__global__ void __launch_bounds__(kDkvThreads, 1)
sap_bwd_dkv_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapDO,
                   const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV,
                   const TileDesc* __restrict__ tiles, const SegDesc* __restrict__ segs,
                   const int32_t* __restrict__ cu, int n_docs, const float* __restrict__ lse,
                   const float* __restrict__ dsum, __nv_bfloat16* __restrict__ dk, __nv_bfloat16* __restrict__ dv,
                   int n_tokens, int n_q_heads, int n_kv_heads, float scale, float scale_log2) {
  using L = DkvSmem<D>;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = smem_raw;
  if (smem_u32(smem) & 1023u) __trap();
  const uint32_t s0 = smem_u32(smem);
  const uint32_t sK = s0 + L::kOffK, sV = s0 + L::kOffV, sQ = s0 + L::kOffQ, sDO = s0 + L::kOffDO;
  float* stat = reinterpret_cast<float*>(smem + L::kOffStat);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::kBarOffset);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::kBarOffset + 192);
  const uint32_t bar_kv_full = smem_u32(bars + 0), bar_qdo_full = smem_u32(bars + 1), bar_qdo_empty = smem_u32(bars + 4),
                 bar_stat_full = smem_u32(bars + 7), bar_stat_empty = smem_u32(bars + 10),
                 bar_s_full = smem_u32(bars + 13), bar_p_full = smem_u32(bars + 15), bar_acc_full = smem_u32(bars + 17);

  // logical warp id: service warps (0-3) are the physically last four (see sap_fwd.cuh)
  const int warp = ((threadIdx.x >> 5) + 4) % (kDkvThreads / 32), lane = threadIdx.x & 31;
  int tile_idx, hk;
  kv_block_coords(n_kv_heads, tile_idx, hk);
  const int g = n_q_heads / n_kv_heads;
  const TileDesc td = tiles[tile_idx];

  if (threadIdx.x == 0) {
    mbar_init(bar_kv_full, 1);
    for (int i = 0; i < kDkvStages; ++i) {
      mbar_init(bar_qdo_full + 8 * i, 1); mbar_init(bar_qdo_empty + 8 * i, 1);
      mbar_init(bar_stat_full + 8 * i, 32); mbar_init(bar_stat_empty + 8 * i, 128 * kDkvParts);
    }
    for (int i = 0; i < 2; ++i) { mbar_init(bar_s_full + 8 * i, 1); mbar_init(bar_p_full + 8 * i, 128 * kDkvParts); }
    mbar_init(bar_acc_full, 1);
    fence_mbar_init();
    tma_prefetch_desc(&mapQ); tma_prefetch_desc(&mapDO); tma_prefetch_desc(&mapK); tma_prefetch_desc(&mapV);
  }
  if (warp == 1) { tmem_alloc(smem_u32(tmem_slot), 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t tDK = tmem, tDV = tmem + 128, tBuf = tmem + 256;

  int iters_per_head = 0;
  for (int s = td.seg_begin; s < td.seg_end; ++s) iters_per_head += (segs[s].t_end - segs[s].t_begin + kBwdN - 1) / kBwdN;
  const int n_iters = iters_per_head * g;

  if (warp == 0) {
    // ------------------------------------------------------------------ TMA producer
    if (n_iters > 0 && elect_one()) {
      mbar_expect_tx(bar_kv_full, 2 * L::kKVBytes);
#pragma unroll
      for (int b = 0; b < L::kBoxes; ++b) {
        tma_load_2d(sK + b * L::kKVBox, &mapK, hk * D + b * 64, td.row0, bar_kv_full);
        tma_load_2d(sV + b * L::kKVBox, &mapV, hk * D + b * 64, td.row0, bar_kv_full);
      }
      int i = 0;
      for (int hq = 0; hq < g; ++hq) {
        const int h = hk * g + hq;
        for (int s = td.seg_begin; s < td.seg_end; ++s) {
          const int t_begin = segs[s].t_begin, t_end = segs[s].t_end;
          for (int t0 = t_begin; t0 < t_end; t0 += kBwdN, ++i) {
            const int st = i % kDkvStages;
            mbar_wait(bar_qdo_empty + 8 * st, ((i / kDkvStages) & 1) ^ 1);
            mbar_expect_tx(bar_qdo_full + 8 * st, 2 * L::kQBytes);
#pragma unroll
            for (int b = 0; b < L::kBoxes; ++b) {
              tma_load_2d(sQ + st * L::kQBytes + b * L::kQBox, &mapQ, h * D + b * 64, t0, bar_qdo_full + 8 * st);
              tma_load_2d(sDO + st * L::kQBytes + b * L::kQBox, &mapDO, h * D + b * 64, t0, bar_qdo_full + 8 * st);
            }
          }
        }
      }
    }
  } else if (warp == 2 || warp == 3) {
    // ------------------------------------------------------------------ per-row LSE (log2 domain) and D loaders
    // two warps take alternate iterations, so each has two iteration times to cover the global-load latency
    int i = 0;
    for (int hq = 0; hq < g; ++hq) {
      const int h = hk * g + hq;
      const float* lse_h = lse + static_cast<size_t>(h) * n_tokens;
      const float* dsum_h = dsum + static_cast<size_t>(h) * n_tokens;
      for (int s = td.seg_begin; s < td.seg_end; ++s) {
        const int t_begin = segs[s].t_begin, t_end = segs[s].t_end;
        for (int t0 = t_begin; t0 < t_end; t0 += kBwdN, ++i) {
          if ((i & 1) != (warp & 1)) continue;
          const int st = i % kDkvStages;
          float a[2], b[2];
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            const int t = t0 + lane + 32 * j;
            a[j] = t < n_tokens ? __ldg(lse_h + t) * kLog2e : CUDART_INF_F;
            b[j] = t < n_tokens ? __ldg(dsum_h + t) : 0.f;
          }
          mbar_wait(bar_stat_empty + 8 * st, ((i / kDkvStages) & 1) ^ 1);
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            stat[st * 128 + lane + 32 * j] = a[j];
            stat[st * 128 + 64 + lane + 32 * j] = b[j];
          }
          mbar_arrive(bar_stat_full + 8 * st);
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------ tcgen05 issuer: one elected thread runs
    // the whole loop (no per-iteration warp sync / election); stage and phase counters are incremental
    if (n_iters > 0 && elect_one()) {
      constexpr uint32_t idesc_s = make_idesc_bf16(128, kBwdN, 0, 0);  // S^T, dP^T [128x64]: K-major x K-major
      constexpr uint32_t idesc_acc = make_idesc_bf16(128, D, 0, 1);    // dV, dK [128xD]: TMEM x MN-major
      const uint64_t dK0 = make_smem_desc(sK, 16, 1024), dV0 = make_smem_desc(sV, 16, 1024);
      const uint64_t dQk0 = make_smem_desc(sQ, 16, 1024), dDOk0 = make_smem_desc(sDO, 16, 1024);          // K-major views
      const uint64_t dQm0 = make_smem_desc(sQ, L::kQBox, 1024), dDOm0 = make_smem_desc(sDO, L::kQBox, 1024);  // MN-major views
      mbar_wait(bar_kv_full, 0);
      int st_i = 0, ph_i = 0, st_j = 0;
      for (int i = 0; i <= n_iters; ++i) {
        if (i < n_iters) {
          const int b = i & 1;
          const uint32_t tST = tBuf + 128 * b, tDPT = tST + 64;
          SAP_STAMP(i, 0);
          mbar_wait(bar_qdo_full + 8 * st_i, ph_i);
          tc_fence_after();
          SAP_STAMP(i, 1);
          const uint64_t dq = desc_add(dQk0, st_i * L::kQBytes), ddo = desc_add(dDOk0, st_i * L::kQBytes);
#pragma unroll
          for (int k = 0; k < D / 16; ++k)
            umma_ss(tST, desc_add(dK0, (k / 4) * L::kKVBox + (k % 4) * 32), desc_add(dq, (k / 4) * L::kQBox + (k % 4) * 32), idesc_s, k > 0);
#pragma unroll
          for (int k = 0; k < D / 16; ++k)
            umma_ss(tDPT, desc_add(dV0, (k / 4) * L::kKVBox + (k % 4) * 32), desc_add(ddo, (k / 4) * L::kQBox + (k % 4) * 32), idesc_s, k > 0);
          umma_commit(bar_s_full + 8 * b);
          SAP_STAMP(i, 2);
          if (++st_i == kDkvStages) { st_i = 0; ph_i ^= 1; }
        }
        if (i > 0) {
          const int j = i - 1, b = j & 1;
          const uint32_t tPT = tBuf + 128 * b, tDST = tPT + 64;
          SAP_STAMP(j, 5);
          mbar_wait(bar_p_full + 8 * b, (j >> 1) & 1);
          tc_fence_after();
          SAP_STAMP(j, 3);
          const uint64_t dq = desc_add(dQm0, st_j * L::kQBytes), ddo = desc_add(dDOm0, st_j * L::kQBytes);
#pragma unroll
          for (int k = 0; k < kBwdN / 16; ++k)  // the bf16 of q rows [16k,16k+16) sit in the 8 columns at 16k
            umma_ts(tDV, tPT + k * 16, desc_add(ddo, k * 2048), idesc_acc, (j > 0 || k > 0) ? 1u : 0u);
#pragma unroll
          for (int k = 0; k < kBwdN / 16; ++k)
            umma_ts(tDK, tDST + k * 16, desc_add(dq, k * 2048), idesc_acc, (j > 0 || k > 0) ? 1u : 0u);
          umma_commit(bar_qdo_empty + 8 * st_j);
          SAP_STAMP(j, 4);
          if (j == n_iters - 1) umma_commit(bar_acc_full);
          if (++st_j == kDkvStages) st_j = 0;
        }
      }
    }
  } else if (warp >= 4) {
    // ------------------------------------------------------------------ compute: P^T, dS^T; epilogue
    const int quarter = warp & 3, part = (warp - 4) >> 2;
    const int r = quarter * 32 + lane;
    const int srow = td.row0 + r;                        // key index owned by this thread
    const bool valid = r < td.rows;
    const uint32_t lane_base = static_cast<uint32_t>(quarter * 32) << 16;
    const int32_t doc_hi = valid ? doc_end_of(cu, n_docs, srow) : 0;
    int i = 0;
    for (int hq = 0; hq < g; ++hq) {
      for (int s = td.seg_begin; s < td.seg_end; ++s) {
        const SegDesc sd = segs[s];
        int lo = max(srow, sd.q_lo), hi = min(doc_hi, sd.q_hi);  // rows t that see key srow: [lo, hi)
        if (!valid || srow < sd.kv_lo || srow >= sd.kv_hi) { lo = 0; hi = 0; }
        for (int t0 = sd.t_begin; t0 < sd.t_end; t0 += kBwdN, ++i) {
          const int st = i % kDkvStages, b = i & 1;
          const uint32_t tST = tBuf + 128 * b + lane_base + kDkvCols * part, tDPT = tST + 64;
          const int tc = t0 + kDkvCols * part;  // first q row of this warp's column part
          if (warp == 4 && lane == 0) SAP_STAMP(i, 8);
          mbar_wait(bar_stat_full + 8 * st, (i / kDkvStages) & 1);
          if (warp == 4 && lane == 0) SAP_STAMP(i, 9);
          mbar_wait(bar_s_full + 8 * b, (i >> 1) & 1);
          tc_fence_after();
          if (lane == 0) SAP_STAMP(i, 16 + warp - 4);
          const bool need_mask = __any_sync(0xffffffffu, (tc < lo) || (tc + kDkvCols > hi));
          uint32_t sv[kDkvCols], dp[kDkvCols];
          tmem_ld16(tST, sv);
          tmem_ld16(tDPT, dp);
          const float4* l4 = reinterpret_cast<const float4*>(stat + st * 128 + kDkvCols * part);
          const float4* d4 = reinterpret_cast<const float4*>(stat + st * 128 + 64 + kDkvCols * part);
          tmem_wait_ld();
          if (warp == 4 && lane == 0) SAP_STAMP(i, 11);
          if (need_mask) {  // boundary tiles only: masked scores become -inf, so P = 2^-inf = 0 and dS = 0
#pragma unroll
            for (int idx = 0; idx < kDkvCols; ++idx) {
              const int t = tc + idx;
              if (!(t >= lo && t < hi)) sv[idx] = 0xff800000u;
            }
          }
          uint32_t pk[kDkvCols / 2], dsk[kDkvCols / 2];
#pragma unroll
          for (int q4 = 0; q4 < kDkvCols / 4; ++q4) {
            const float4 lv = l4[q4], dvv = d4[q4];
            const float ls[4] = {lv.x, lv.y, lv.z, lv.w}, dd[4] = {dvv.x, dvv.y, dvv.z, dvv.w};
            float p[4], ds[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const int idx = q4 * 4 + e;
              p[e] = ex2_approx(fmaf(__uint_as_float(sv[idx]), scale_log2, -ls[e]));
              ds[e] = p[e] * (__uint_as_float(dp[idx]) - dd[e]);
            }
            pk[q4 * 2] = pack_bf16x2(p[0], p[1]); pk[q4 * 2 + 1] = pack_bf16x2(p[2], p[3]);
            dsk[q4 * 2] = pack_bf16x2(ds[0], ds[1]); dsk[q4 * 2 + 1] = pack_bf16x2(ds[2], ds[3]);
          }
          if (lane == 0) SAP_STAMP(i, 48 + warp - 4);
          tmem_st8(tST, pk);     // bf16 P^T over the S^T columns this warp has just read
          tmem_st8(tDPT, dsk);   // bf16 dS^T over its dP^T columns
          tmem_wait_st();
          tc_fence_before();
          if (lane == 0) SAP_STAMP(i, 32 + warp - 4);
          mbar_arrive(bar_p_full + 8 * b);
          mbar_arrive(bar_stat_empty + 8 * st);
        }
      }
    }
    if (n_iters > 0) {
      mbar_wait(bar_acc_full, 0);
      tc_fence_after();
    }
    // parts 0,1 write the two column halves of dK (scaled), parts 2,3 those of dV
    const bool is_dk = part < 2;
    const int chalf = part & 1;
    const uint32_t tAcc = (is_dk ? tDK : tDV) + lane_base + chalf * (D / 2);
    const float mul = is_dk ? scale : 1.f;
    __nv_bfloat16* dst_base = (is_dk ? dk : dv) + (static_cast<size_t>(srow) * n_kv_heads + hk) * D + chalf * (D / 2);
#pragma unroll
    for (int c = 0; c < D / 64; ++c) {
      uint32_t v[32];
      if (n_iters > 0) {
        tmem_ld32(tAcc + c * 32, v);
        tmem_wait_ld();
      } else {
#pragma unroll
        for (int e = 0; e < 32; ++e) v[e] = 0u;
      }
      if (valid) {
        uint4* dst = reinterpret_cast<uint4*>(dst_base + c * 32);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          uint4 w;
          w.x = pack_bf16x2(__uint_as_float(v[8 * e + 0]) * mul, __uint_as_float(v[8 * e + 1]) * mul);
          w.y = pack_bf16x2(__uint_as_float(v[8 * e + 2]) * mul, __uint_as_float(v[8 * e + 3]) * mul);
          w.z = pack_bf16x2(__uint_as_float(v[8 * e + 4]) * mul, __uint_as_float(v[8 * e + 5]) * mul);
          w.w = pack_bf16x2(__uint_as_float(v[8 * e + 6]) * mul, __uint_as_float(v[8 * e + 7]) * mul);
          dst[e] = w;
        }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, 512);
}

}  // namespace sap

#include "sap_bwd_dq.cuh"
