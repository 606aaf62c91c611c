// Fused backward kernel: dK, dV AND dQ from one pass over the visible (key tile, row tile) pairs,
// 5 GEMMs per pair instead of the 7 of the split form (sap_bwd_dkv_kernel + sap_bwd_dq_kernel).
// (Table 1 tensors do / dq / dkv; fwd+bwd is what the paper times, :173.)
//
// One CTA = one 128-row K/V tile x one kv-head, one CTA per SM, 896 threads:
//   service warps: TMA producer, tcgen05 issuer (one elected thread each), two LSE/D loader warps;
//   16 compute warps: warp w owns TMEM lane quarter w%4 and column part (w-4)/4 (16 of the 64 streamed q rows);
//   8 drain warps (two warpgroups, 32 of the 64 q rows each): move each finished dQ^T tile from TMEM to registers,
//   release the TMEM columns, then add the tile into the global fp32 accumulator.
// Per streamed 64-row Q/dO tile of a q-head of the group (KV-stationary, keys on TMEM lanes):
//   S^T  = K Q^T, dP^T = V dO^T            (smem x smem -> TMEM score buffer b, [128 keys x 64 rows] fp32 each)
//   P^T  = 2^(scale*log2e*S^T - LSE),  dS^T = P^T (dP^T - D)        (compute warps)
//        P^T  bf16 -> TMEM over the S^T columns (A operand of dV)
//        dS^T bf16 -> shared memory, 128B-swizzled [128 keys x 64 rows] (A operand of dK, B operand of dQ^T)
//   dQ^T = K^T dS^T   [128 (d) x 64 rows]  (K as MN-major A, dS^T as MN-major B) -> TMEM over the dP^T columns
//   dV  += P^T dO, dK += dS^T Q            (accumulate over all rows and the Hq/Hkv q-heads of the group)
//   dQ^T is drained by the drain warps with red.global.add.f32 into the fp32 workspace dq_acc [N,Hq,d]
//   (lane = d index, so every warp-level reduction is one coalesced 128-byte line), unscaled.
// sap_bwd_post_kernel (a7) then writes dq = bf16(scale * dq_acc).
//
// TMEM (512 columns): [0,128) dK | [128,256) dV | two score buffers b at 256+128b: [0,64) S^T -> P^T, [64,128) dP^T -> dQ^T.
#pragma once
#include <cuda_bf16.h>
#include <math_constants.h>
#include "sap_bwd.cuh"

namespace sap {

constexpr int kFusedParts = 4;
constexpr int kFusedDrainGroups = 2;
constexpr int kFusedThreads = 128 + 128 * kFusedParts + 128 * kFusedDrainGroups;  // service + compute + drain warpgroups
// setmaxnreg split of the 896 x 72 register pool: 512*88 (compute) + 128*56 (service) + 256*48 (drain)
constexpr int kFusedRegsCompute = 88, kFusedRegsService = 56, kFusedRegsDrain = 48;
constexpr int kFusedCols = kBwdN / kFusedParts;  // q rows (TMEM columns) per compute warp
constexpr int kFusedStages = 3;

template <int D>
struct FusedSmem {
  static constexpr int kKVBytes = kTile * D * 2;   // K or V, 128 rows
  static constexpr int kQBytes = kBwdN * D * 2;    // Q or dO stage, 64 rows
  static constexpr int kKVBox = kTile * 128;
  static constexpr int kQBox = kBwdN * 128;
  static constexpr int kBoxes = D / 64;
  static constexpr int kDSBytes = kTile * kBwdN * 2;  // dS^T bf16 [128 keys x 64 rows]
  static constexpr int kOffK = 0, kOffV = kKVBytes, kOffQ = 2 * kKVBytes, kOffDO = kOffQ + kFusedStages * kQBytes;
  static constexpr int kOffDS = kOffDO + kFusedStages * kQBytes;  // two buffers
  static constexpr int kOffStat = kOffDS + 2 * kDSBytes;          // [stage][2][64] floats
  static constexpr int kBarOffset = kOffStat + kFusedStages * 512;
  static constexpr int kTotal = kBarOffset + 256;
};

__device__ __forceinline__ void red_add_f32(float* addr, float v) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}

template <int D>
__global__ void __launch_bounds__(kFusedThreads, 1)
sap_bwd_fused_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapDO,
                     const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV,
                     const TileDesc* __restrict__ tiles, const SegDesc* __restrict__ segs,
                     const int32_t* __restrict__ cu, int n_docs, const float* __restrict__ lse,
                     const float* __restrict__ dsum, float* __restrict__ dq_acc, __nv_bfloat16* __restrict__ dk,
                     __nv_bfloat16* __restrict__ dv, int n_tokens, int n_q_heads, int n_kv_heads, float scale,
                     float scale_log2) {
  using L = FusedSmem<D>;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = smem_raw;
  if (smem_u32(smem) & 1023u) __trap();
  const uint32_t s0 = smem_u32(smem);
  const uint32_t sK = s0 + L::kOffK, sV = s0 + L::kOffV, sQ = s0 + L::kOffQ, sDO = s0 + L::kOffDO, sDS = s0 + L::kOffDS;
  float* stat = reinterpret_cast<float*>(smem + L::kOffStat);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::kBarOffset);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::kBarOffset + 240);
  const uint32_t bar_kv_full = smem_u32(bars + 0), bar_qdo_full = smem_u32(bars + 1), bar_qdo_empty = smem_u32(bars + 4),
                 bar_stat_full = smem_u32(bars + 7), bar_stat_empty = smem_u32(bars + 10),
                 bar_s_full = smem_u32(bars + 13), bar_p_full = smem_u32(bars + 15), bar_acc_full = smem_u32(bars + 17),
                 bar_dq_full = smem_u32(bars + 18), bar_dq_empty = smem_u32(bars + 20);

  // logical warp id: service warps (0-3) are the physically last four (see sap_fwd.cuh)
  const int warp = ((threadIdx.x >> 5) + 4) % (kFusedThreads / 32), lane = threadIdx.x & 31;
  int tile_idx, hk;
  kv_block_coords(n_kv_heads, tile_idx, hk);
  const int g = n_q_heads / n_kv_heads;
  const TileDesc td = tiles[tile_idx];

  if (threadIdx.x == 0) {
    mbar_init(bar_kv_full, 1);
    for (int i = 0; i < kFusedStages; ++i) {
      mbar_init(bar_qdo_full + 8 * i, 1); mbar_init(bar_qdo_empty + 8 * i, 1);
      mbar_init(bar_stat_full + 8 * i, 32); mbar_init(bar_stat_empty + 8 * i, 128 * kFusedParts);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(bar_s_full + 8 * i, 1); mbar_init(bar_p_full + 8 * i, 128 * kFusedParts);
      mbar_init(bar_dq_full + 8 * i, 1); mbar_init(bar_dq_empty + 8 * i, 128 * kFusedDrainGroups);
    }
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

  if (warp < 4) reg_dealloc<kFusedRegsService>();
  if (warp == 0) {
    // ------------------------------------------------------------------ TMA producer
    if (n_iters > 0 && elect_one()) {
      mbar_expect_tx(bar_kv_full, 2 * L::kKVBytes);
#pragma unroll
      for (int b = 0; b < L::kBoxes; ++b) {
        tma_load_2d(sK + b * L::kKVBox, &mapK, hk * D + b * 64, td.row0, bar_kv_full);
        tma_load_2d(sV + b * L::kKVBox, &mapV, hk * D + b * 64, td.row0, bar_kv_full);
      }
      int st = 0, ph = 1;  // empty barriers: the first pass over the ring must not block
      for (int hq = 0; hq < g; ++hq) {
        const int h = hk * g + hq;
        for (int s = td.seg_begin; s < td.seg_end; ++s) {
          const int t_begin = segs[s].t_begin, t_end = segs[s].t_end;
          for (int t0 = t_begin; t0 < t_end; t0 += kBwdN) {
            mbar_wait(bar_qdo_empty + 8 * st, ph);
            mbar_expect_tx(bar_qdo_full + 8 * st, 2 * L::kQBytes);
#pragma unroll
            for (int b = 0; b < L::kBoxes; ++b) {
              tma_load_2d(sQ + st * L::kQBytes + b * L::kQBox, &mapQ, h * D + b * 64, t0, bar_qdo_full + 8 * st);
              tma_load_2d(sDO + st * L::kQBytes + b * L::kQBox, &mapDO, h * D + b * 64, t0, bar_qdo_full + 8 * st);
            }
            if (++st == kFusedStages) { st = 0; ph ^= 1; }
          }
        }
      }
    }
  } else if (warp == 2 || warp == 3) {
    // ------------------------------------------------------------------ per-row LSE (log2 domain) and D loaders
    int i = 0;
    for (int hq = 0; hq < g; ++hq) {
      const int h = hk * g + hq;
      const float* lse_h = lse + static_cast<size_t>(h) * n_tokens;
      const float* dsum_h = dsum + static_cast<size_t>(h) * n_tokens;
      for (int s = td.seg_begin; s < td.seg_end; ++s) {
        const int t_begin = segs[s].t_begin, t_end = segs[s].t_end;
        for (int t0 = t_begin; t0 < t_end; t0 += kBwdN, ++i) {
          if ((i & 1) != (warp & 1)) continue;
          const int st = i % kFusedStages;
          float a[2], b[2];
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            const int t = t0 + lane + 32 * j;
            a[j] = t < n_tokens ? __ldg(lse_h + t) * kLog2e : CUDART_INF_F;
            b[j] = t < n_tokens ? __ldg(dsum_h + t) : 0.f;
          }
          mbar_wait(bar_stat_empty + 8 * st, ((i / kFusedStages) & 1) ^ 1);
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
    // ------------------------------------------------------------------ tcgen05 issuer (one elected thread)
    if (n_iters > 0 && elect_one()) {
      constexpr uint32_t idesc_s = make_idesc_bf16(128, kBwdN, 0, 0);   // S^T, dP^T [128x64]: K-major x K-major
      constexpr uint32_t idesc_dv = make_idesc_bf16(128, D, 0, 1);      // dV [128xD]: P^T (TMEM) x dO (MN-major)
      constexpr uint32_t idesc_dk = make_idesc_bf16(128, D, 0, 1);      // dK [128xD]: dS^T (smem, K-major) x Q (MN-major)
      constexpr uint32_t idesc_dq = make_idesc_bf16(128, kBwdN, 1, 1);  // dQ^T [128x64]: K (MN-major A) x dS^T (MN-major B)
      const uint64_t dK0 = make_smem_desc(sK, 16, 1024), dV0 = make_smem_desc(sV, 16, 1024);
      const uint64_t dKm0 = make_smem_desc(sK, L::kKVBox, 1024);                                           // K as MN-major A (M = d)
      const uint64_t dQk0 = make_smem_desc(sQ, 16, 1024), dDOk0 = make_smem_desc(sDO, 16, 1024);            // K-major views
      const uint64_t dQm0 = make_smem_desc(sQ, L::kQBox, 1024), dDOm0 = make_smem_desc(sDO, L::kQBox, 1024);  // MN-major views
      const uint64_t dDSk0 = make_smem_desc(sDS, 16, 1024);          // dS^T as K-major A (K = q rows)
      const uint64_t dDSm0 = make_smem_desc(sDS, L::kDSBytes, 1024);  // dS^T as MN-major B (N = q rows: one 64-wide atom)
      mbar_wait(bar_kv_full, 0);
      int st_i = 0, ph_i = 0, st_j = 0;
      for (int i = 0; i <= n_iters; ++i) {
        if (i < n_iters) {
          const int b = i & 1;
          const uint32_t tST = tBuf + 128 * b, tDPT = tST + 64;
          mbar_wait(bar_qdo_full + 8 * st_i, ph_i);
          tc_fence_after();
          const uint64_t dq = desc_add(dQk0, st_i * L::kQBytes), ddo = desc_add(dDOk0, st_i * L::kQBytes);
#pragma unroll
          for (int k = 0; k < D / 16; ++k)
            umma_ss(tST, desc_add(dK0, (k / 4) * L::kKVBox + (k % 4) * 32), desc_add(dq, (k / 4) * L::kQBox + (k % 4) * 32), idesc_s, k > 0);
          if (i >= 2) {  // dQ^T of tile i-2 must have been drained from the dP^T columns
            mbar_wait(bar_dq_empty + 8 * b, ((i >> 1) - 1) & 1);
            tc_fence_after();
          }
#pragma unroll
          for (int k = 0; k < D / 16; ++k)
            umma_ss(tDPT, desc_add(dV0, (k / 4) * L::kKVBox + (k % 4) * 32), desc_add(ddo, (k / 4) * L::kQBox + (k % 4) * 32), idesc_s, k > 0);
          umma_commit(bar_s_full + 8 * b);
          if (++st_i == kFusedStages) { st_i = 0; ph_i ^= 1; }
        }
        if (i > 0) {
          const int j = i - 1, b = j & 1;
          const uint32_t tPT = tBuf + 128 * b, tDQT = tPT + 64;
          mbar_wait(bar_p_full + 8 * b, (j >> 1) & 1);
          tc_fence_after();
          const uint64_t dq = desc_add(dQm0, st_j * L::kQBytes), ddo = desc_add(dDOm0, st_j * L::kQBytes);
          const uint64_t dsk = desc_add(dDSk0, b * L::kDSBytes), dsm = desc_add(dDSm0, b * L::kDSBytes);
          // dQ^T first: its drain then overlaps the dV / dK MMAs
#pragma unroll
          for (int k = 0; k < kTile / 16; ++k)  // 16 keys per MMA: two 8-row groups (SBO 1024 B)
            umma_ss(tDQT, desc_add(dKm0, k * 2048), desc_add(dsm, k * 2048), idesc_dq, k > 0);
          umma_commit(bar_dq_full + 8 * b);
#pragma unroll
          for (int k = 0; k < kBwdN / 16; ++k)  // the bf16 of q rows [16k,16k+16) sit in the 8 columns at 16k
            umma_ts(tDV, tPT + k * 16, desc_add(ddo, k * 2048), idesc_dv, (j > 0 || k > 0) ? 1u : 0u);
#pragma unroll
          for (int k = 0; k < kBwdN / 16; ++k)
            umma_ss(tDK, desc_add(dsk, k * 32), desc_add(dq, k * 2048), idesc_dk, (j > 0 || k > 0) ? 1u : 0u);
          umma_commit(bar_qdo_empty + 8 * st_j);
          if (j == n_iters - 1) umma_commit(bar_acc_full);
          if (++st_j == kFusedStages) st_j = 0;
        }
      }
    }
  } else if (warp >= 4 + 4 * kFusedParts) {
    // ------------------------------------------------------------------ drain: dQ^T (TMEM) -> dq_acc (global, fp32 red)
    reg_dealloc<kFusedRegsDrain>();
    const int quarter = warp & 3, dpart = (warp - 4 - 4 * kFusedParts) >> 2;
    constexpr int kCols = kBwdN / kFusedDrainGroups;      // q rows (TMEM columns) per drain warp
    const int r = quarter * 32 + lane;                   // dQ^T lane = d index
    const uint32_t lane_base = static_cast<uint32_t>(quarter * 32) << 16;
    const bool drain_lane = r < D;                        // for D = 64 the upper 64 lanes hold don't-care values
    const size_t row_stride = static_cast<size_t>(n_q_heads) * D;
    int j = 0;
    for (int hq = 0; hq < g; ++hq) {
      const int h = hk * g + hq;
      for (int s = td.seg_begin; s < td.seg_end; ++s) {
        const int t_begin = segs[s].t_begin, t_end = segs[s].t_end;
        for (int t0 = t_begin; t0 < t_end; t0 += kBwdN, ++j) {
          const int b = j & 1;
          const int tq = t0 + kCols * dpart;
          float* dst = dq_acc + (static_cast<size_t>(tq) * n_q_heads + h) * D + r;
          mbar_wait(bar_dq_full + 8 * b, (j >> 1) & 1);
          tc_fence_after();
          uint32_t v[kCols];
          tmem_ld32(tBuf + 128 * b + 64 + lane_base + kCols * dpart, v);
          tmem_wait_ld();
          tc_fence_before();
          mbar_arrive(bar_dq_empty + 8 * b);  // the dP^T / dQ^T columns of buffer b are free again
          if (drain_lane) {
            if (tq + kCols <= n_tokens) {
#pragma unroll
              for (int c = 0; c < kCols; ++c) { red_add_f32(dst, __uint_as_float(v[c])); dst += row_stride; }
            } else {
#pragma unroll
              for (int c = 0; c < kCols; ++c) {
                if (tq + c < n_tokens) red_add_f32(dst, __uint_as_float(v[c]));
                dst += row_stride;
              }
            }
          }
        }
      }
    }
  } else if (warp >= 4) {
    // ------------------------------------------------------------------ compute: P^T, dS^T; epilogue
    reg_alloc<kFusedRegsCompute>();
    const int quarter = warp & 3, part = (warp - 4) >> 2;
    const int r = quarter * 32 + lane;
    const int srow = td.row0 + r;                        // key index owned by this thread
    const bool valid = r < td.rows;
    const uint32_t lane_base = static_cast<uint32_t>(quarter * 32) << 16;
    const int32_t doc_hi = valid ? doc_end_of(cu, n_docs, srow) : 0;
    // this thread's two 16-byte chunks of the dS^T row (128B swizzle: chunk c of row r sits at c ^ (r & 7))
    uint8_t* ds_row = smem + L::kOffDS + (r >> 3) * 1024 + (r & 7) * 128;
    const int ch0 = ((2 * part) ^ (r & 7)) << 4, ch1 = ((2 * part + 1) ^ (r & 7)) << 4;

    int i = 0;
    for (int hq = 0; hq < g; ++hq) {
      for (int s = td.seg_begin; s < td.seg_end; ++s) {
        const SegDesc sd = segs[s];
        int lo = max(srow, sd.q_lo), hi = min(doc_hi, sd.q_hi);  // rows t that see key srow: [lo, hi)
        if (!valid || srow < sd.kv_lo || srow >= sd.kv_hi) { lo = 0; hi = 0; }
        for (int t0 = sd.t_begin; t0 < sd.t_end; t0 += kBwdN, ++i) {
          const int st = i % kFusedStages, b = i & 1;
          const uint32_t tST = tBuf + 128 * b + lane_base + kFusedCols * part, tDPT = tST + 64;
          const int tc = t0 + kFusedCols * part;  // first q row of this warp's column part
          mbar_wait(bar_stat_full + 8 * st, (i / kFusedStages) & 1);
          mbar_wait(bar_s_full + 8 * b, (i >> 1) & 1);
          tc_fence_after();
          const bool need_mask = __any_sync(0xffffffffu, (tc < lo) || (tc + kFusedCols > hi));
          uint32_t sv[kFusedCols], dp[kFusedCols];
          tmem_ld16(tST, sv);
          tmem_ld16(tDPT, dp);
          const float4* l4 = reinterpret_cast<const float4*>(stat + st * 128 + kFusedCols * part);
          const float4* d4 = reinterpret_cast<const float4*>(stat + st * 128 + 64 + kFusedCols * part);
          tmem_wait_ld();
          if (need_mask) {  // boundary tiles only: masked scores become -inf, so P = 2^-inf = 0 and dS = 0
#pragma unroll
            for (int idx = 0; idx < kFusedCols; ++idx) {
              const int t = tc + idx;
              if (!(t >= lo && t < hi)) sv[idx] = 0xff800000u;
            }
          }
          uint32_t pk[kFusedCols / 2], dsk[kFusedCols / 2];
#pragma unroll
          for (int q4 = 0; q4 < kFusedCols / 4; ++q4) {
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
          tmem_st8(tST, pk);     // bf16 P^T over the S^T columns this warp has just read
          uint8_t* ds_dst = ds_row + b * L::kDSBytes;
          *reinterpret_cast<uint4*>(ds_dst + ch0) = make_uint4(dsk[0], dsk[1], dsk[2], dsk[3]);
          *reinterpret_cast<uint4*>(ds_dst + ch1) = make_uint4(dsk[4], dsk[5], dsk[6], dsk[7]);
          tmem_wait_st();
          tc_fence_before();
          fence_proxy_async_smem();  // the dS^T stores must be visible to the tensor core's (async proxy) reads
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

// ------------------------------------------------------------------------------------------------
// a7: dq = bf16(scale * dq_acc).  HBM-bound: 4 B read + 2 B written per element, 32-byte loads / 16-byte stores.
// ------------------------------------------------------------------------------------------------
constexpr int kPostThreads = 256;

__global__ void __launch_bounds__(kPostThreads)
sap_bwd_post_kernel(const float* __restrict__ dq_acc, __nv_bfloat16* __restrict__ dq, int64_t n_elems8, float scale) {
  const int64_t stride = static_cast<int64_t>(gridDim.x) * blockDim.x;
  for (int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; i < n_elems8; i += stride) {
    const float4 a = __ldcs(reinterpret_cast<const float4*>(dq_acc) + 2 * i);
    const float4 b = __ldcs(reinterpret_cast<const float4*>(dq_acc) + 2 * i + 1);
    uint4 w;
    w.x = pack_bf16x2(a.x * scale, a.y * scale); w.y = pack_bf16x2(a.z * scale, a.w * scale);
    w.z = pack_bf16x2(b.x * scale, b.y * scale); w.w = pack_bf16x2(b.z * scale, b.w * scale);
    reinterpret_cast<uint4*>(dq)[i] = w;
  }
}

}  // namespace sap
