// dQ kernel (included by sap_bwd.cuh).  One CTA = one 128-row Q tile x one q-head, ONE CTA per SM, 640 threads:
//   service warps: TMA producer, tcgen05 issuer (one elected thread each);
//   16 compute warps: warp w owns TMEM lane quarter w%4 (= 32 Q rows) and key-column part (w-4)/4 (16 of the 64
//   streamed keys), so every thread handles 16 scores per iteration with its row's LSE and D in registers.
//
// Q and dO are copied once from shared memory into TMEM and used as the A operand of S = Q K^T and dP = dO V^T:
// tcgen05.mma with A in TMEM runs N=64 tiles at the full rate, while the shared-memory A path is bandwidth-bound
// at N=64 (48 instead of 32 cycles per MMA, measured).  The issuer runs one key tile ahead of the compute warps
// (two score buffers), as in the dK/dV kernel.
//
// TMEM (512 columns): [0,128) dQ fp32 | [128,192) Q bf16 | [192,256) dO bf16 | two buffers b at 256+128b:
//   S fp32 [0,64) with dS bf16 written over columns [16p, 16p+8) by the warp of part p; dP fp32 [64,128).
#pragma once

namespace sap {

constexpr int kDqParts = 4;
constexpr int kDqThreads = 128 + 128 * kDqParts;
constexpr int kDqCols = kBwdN / kDqParts;  // keys (TMEM columns) per compute warp
constexpr int kDqStages = 4;               // K/V ring

template <int D>
struct DqSmem {
  static constexpr int kQBytes = kTile * D * 2;   // Q or dO, 128 rows
  static constexpr int kKBytes = kBwdN * D * 2;   // K or V stage, 64 rows
  static constexpr int kQBox = kTile * 128;       // 128 rows x 128 B
  static constexpr int kKBox = kBwdN * 128;       // 64 rows x 128 B
  static constexpr int kBoxes = D / 64;
  static constexpr int kOffQ = 0, kOffDO = kQBytes, kOffK = 2 * kQBytes, kOffV = 2 * kQBytes + kDqStages * kKBytes;
  static constexpr int kBarOffset = kOffV + kDqStages * kKBytes;
  static constexpr int kTotal = kBarOffset + 256;  // dynamic smem base is required to be 1024 B aligned
};

template <int D>
__global__ void __launch_bounds__(kDqThreads, 1)
sap_bwd_dq_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapDO,
                  const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV,
                  const TileDesc* __restrict__ tiles, const SegDesc* __restrict__ segs,
                  const int32_t* __restrict__ cu, int n_docs, const float* __restrict__ lse,
                  const float* __restrict__ dsum, __nv_bfloat16* __restrict__ dq, int n_tokens, int n_q_heads,
                  int n_kv_heads, float scale, float scale_log2) {
  using L = DqSmem<D>;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = smem_raw;
  if (smem_u32(smem) & 1023u) __trap();
  const uint32_t s0 = smem_u32(smem);
  const uint32_t sQ = s0 + L::kOffQ, sDO = s0 + L::kOffDO, sK = s0 + L::kOffK, sV = s0 + L::kOffV;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::kBarOffset);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::kBarOffset + 192);
  const uint32_t bar_q_full = smem_u32(bars + 0), bar_qt_full = smem_u32(bars + 1), bar_kv_full = smem_u32(bars + 2),
                 bar_kv_empty = smem_u32(bars + 6), bar_s_full = smem_u32(bars + 10), bar_ds_full = smem_u32(bars + 12),
                 bar_dq_full = smem_u32(bars + 14);

  // logical warp id: service warps (0-3) are the physically last four (see sap_fwd.cuh)
  const int warp = ((threadIdx.x >> 5) + 4) % (kDqThreads / 32), lane = threadIdx.x & 31;
  int tile_idx, h;
  q_block_coords(n_q_heads, n_kv_heads, tile_idx, h);
  const int hk = h / (n_q_heads / n_kv_heads);
  const TileDesc td = tiles[tile_idx];

  if (threadIdx.x == 0) {
    mbar_init(bar_q_full, 1); mbar_init(bar_qt_full, 128 * kDqParts);
    for (int i = 0; i < kDqStages; ++i) { mbar_init(bar_kv_full + 8 * i, 1); mbar_init(bar_kv_empty + 8 * i, 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(bar_s_full + 8 * i, 1); mbar_init(bar_ds_full + 8 * i, 128 * kDqParts); }
    mbar_init(bar_dq_full, 1);
    fence_mbar_init();
    tma_prefetch_desc(&mapQ); tma_prefetch_desc(&mapDO); tma_prefetch_desc(&mapK); tma_prefetch_desc(&mapV);
  }
  if (warp == 1) { tmem_alloc(smem_u32(tmem_slot), 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t tDQ = tmem, tQ = tmem + 128, tDO = tmem + 192, tBuf = tmem + 256;

  int n_iters = 0;
  for (int s = td.seg_begin; s < td.seg_end; ++s) n_iters += (segs[s].t_end - segs[s].t_begin + kBwdN - 1) / kBwdN;

  if (warp == 0) {
    // ------------------------------------------------------------------ TMA producer
    if (n_iters > 0 && elect_one()) {
      mbar_expect_tx(bar_q_full, 2 * L::kQBytes);
#pragma unroll
      for (int b = 0; b < L::kBoxes; ++b) {
        tma_load_2d(sQ + b * L::kQBox, &mapQ, h * D + b * 64, td.row0, bar_q_full);
        tma_load_2d(sDO + b * L::kQBox, &mapDO, h * D + b * 64, td.row0, bar_q_full);
      }
      int st = 0, ph = 1;  // empty barriers: the first pass over the ring must not block
      for (int s = td.seg_begin; s < td.seg_end; ++s) {
        const int c_begin = segs[s].t_begin, c_end = segs[s].t_end;
        for (int c0 = c_begin; c0 < c_end; c0 += kBwdN) {
          mbar_wait(bar_kv_empty + 8 * st, ph);
          mbar_expect_tx(bar_kv_full + 8 * st, 2 * L::kKBytes);
#pragma unroll
          for (int b = 0; b < L::kBoxes; ++b) {
            tma_load_2d(sK + st * L::kKBytes + b * L::kKBox, &mapK, hk * D + b * 64, c0, bar_kv_full + 8 * st);
            tma_load_2d(sV + st * L::kKBytes + b * L::kKBox, &mapV, hk * D + b * 64, c0, bar_kv_full + 8 * st);
          }
          if (++st == kDqStages) { st = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------ tcgen05 issuer (one elected thread)
    if (n_iters > 0 && elect_one()) {
      constexpr uint32_t idesc_s = make_idesc_bf16(128, kBwdN, 0, 0);  // S, dP [128x64] = A (TMEM) x B (K-major)
      constexpr uint32_t idesc_dq = make_idesc_bf16(128, D, 0, 1);     // dQ [128xD]   = dS (TMEM) x K (MN-major)
      const uint64_t dKk0 = make_smem_desc(sK, 16, 1024), dVk0 = make_smem_desc(sV, 16, 1024);
      const uint64_t dKm0 = make_smem_desc(sK, L::kKBox, 1024);
      mbar_wait(bar_qt_full, 0);
      tc_fence_after();
      int st_i = 0, ph_i = 0, st_j = 0;
      for (int i = 0; i <= n_iters; ++i) {
        if (i < n_iters) {
          const int b = i & 1;
          const uint32_t tS = tBuf + 128 * b, tDP = tS + 64;
          mbar_wait(bar_kv_full + 8 * st_i, ph_i);
          tc_fence_after();
          const uint64_t dk = desc_add(dKk0, st_i * L::kKBytes), dv = desc_add(dVk0, st_i * L::kKBytes);
#pragma unroll
          for (int k = 0; k < D / 16; ++k)
            umma_ts(tS, tQ + k * 8, desc_add(dk, (k / 4) * L::kKBox + (k % 4) * 32), idesc_s, k > 0);
#pragma unroll
          for (int k = 0; k < D / 16; ++k)
            umma_ts(tDP, tDO + k * 8, desc_add(dv, (k / 4) * L::kKBox + (k % 4) * 32), idesc_s, k > 0);
          umma_commit(bar_s_full + 8 * b);
          if (++st_i == kDqStages) { st_i = 0; ph_i ^= 1; }
        }
        if (i > 0) {
          const int j = i - 1, b = j & 1;
          const uint32_t tDS = tBuf + 128 * b;
          mbar_wait(bar_ds_full + 8 * b, (j >> 1) & 1);
          tc_fence_after();
          const uint64_t dk = desc_add(dKm0, st_j * L::kKBytes);
#pragma unroll
          for (int k = 0; k < kBwdN / 16; ++k)  // the bf16 of keys [16k,16k+16) sit in the 8 columns at 16k
            umma_ts(tDQ, tDS + k * 16, desc_add(dk, k * 2048), idesc_dq, (j > 0 || k > 0) ? 1u : 0u);
          umma_commit(bar_kv_empty + 8 * st_j);
          if (j == n_iters - 1) umma_commit(bar_dq_full);
          if (++st_j == kDqStages) st_j = 0;
        }
      }
    }
  } else if (warp >= 4) {
    // ------------------------------------------------------------------ compute warps
    const int quarter = warp & 3, part = (warp - 4) >> 2;
    const int r = quarter * 32 + lane;
    const int t = td.row0 + r;
    const bool valid = r < td.rows;
    const uint32_t lane_base = static_cast<uint32_t>(quarter * 32) << 16;
    const int32_t doc_lo = valid ? doc_start_of(cu, n_docs, t) : 0;
    const float lse2 = valid ? lse[static_cast<size_t>(h) * n_tokens + t] * kLog2e : CUDART_INF_F;
    const float dsum_t = valid ? dsum[static_cast<size_t>(h) * n_tokens + t] : 0.f;
    if (n_iters > 0) {
      // Q and dO rows: 128B-swizzled shared memory -> TMEM A-operand layout (lane = row, column c = elements 2c, 2c+1)
      constexpr int kWords = D / 8;  // 32-bit words (= TMEM columns) per part
      mbar_wait(bar_q_full, 0);
#pragma unroll
      for (int which = 0; which < 2; ++which) {
        const uint8_t* src = smem + (which == 0 ? L::kOffQ : L::kOffDO);
        uint32_t w[kWords];
#pragma unroll
        for (int j = 0; j < kWords / 4; ++j) {
          const int chunk = part * (kWords / 4) + j;           // 16-byte chunk of the row
          const int box = chunk >> 3, cidx = chunk & 7;
          const uint4 v = *reinterpret_cast<const uint4*>(src + box * L::kQBox + r * 128 + ((cidx ^ (r & 7)) << 4));
          w[4 * j + 0] = v.x; w[4 * j + 1] = v.y; w[4 * j + 2] = v.z; w[4 * j + 3] = v.w;
        }
        const uint32_t dst = (which == 0 ? tQ : tDO) + lane_base + part * kWords;
        if constexpr (kWords == 16) tmem_st16(dst, w); else tmem_st8(dst, w);
      }
      tmem_wait_st();
      tc_fence_before();
      mbar_arrive(bar_qt_full);
    }
    int i = 0;
    for (int s = td.seg_begin; s < td.seg_end; ++s) {
      const SegDesc sd = segs[s];
      int lo = max(doc_lo, sd.kv_lo), hi = min(t + 1, sd.kv_hi);  // visible keys of this row: [lo, hi)
      if (!valid || t < sd.q_lo || t >= sd.q_hi) { lo = 0; hi = 0; }
      for (int c0 = sd.t_begin; c0 < sd.t_end; c0 += kBwdN, ++i) {
        const int b = i & 1;
        const uint32_t tS = tBuf + 128 * b + lane_base + kDqCols * part, tDP = tS + 64;
        const int cc = c0 + kDqCols * part;  // first key of this warp's column part
        mbar_wait(bar_s_full + 8 * b, (i >> 1) & 1);
        tc_fence_after();
        const bool need_mask = __any_sync(0xffffffffu, (cc < lo) || (cc + kDqCols > hi));
        uint32_t sv[kDqCols], dp[kDqCols];
        tmem_ld16(tS, sv);
        tmem_ld16(tDP, dp);
        tmem_wait_ld();
        if (need_mask) {  // boundary tiles only: masked scores become -inf => P = 0 => dS = 0
#pragma unroll
          for (int idx = 0; idx < kDqCols; ++idx) {
            const int col = cc + idx;
            if (!(col >= lo && col < hi)) sv[idx] = 0xff800000u;
          }
        }
        uint32_t dsk[kDqCols / 2];
#pragma unroll
        for (int idx = 0; idx < kDqCols; idx += 2) {
          const float p0 = ex2_approx(fmaf(__uint_as_float(sv[idx]), scale_log2, -lse2));
          const float p1 = ex2_approx(fmaf(__uint_as_float(sv[idx + 1]), scale_log2, -lse2));
          dsk[idx >> 1] = pack_bf16x2(p0 * (__uint_as_float(dp[idx]) - dsum_t), p1 * (__uint_as_float(dp[idx + 1]) - dsum_t));
        }
        tmem_st8(tS, dsk);  // bf16 dS over the S columns this warp has just read
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(bar_ds_full + 8 * b);
      }
    }
    if (n_iters > 0) {
      mbar_wait(bar_dq_full, 0);
      tc_fence_after();
    }
    // each part writes D/4 columns of its rows
    constexpr int kOutCols = D / 4;
    const size_t row_off = (static_cast<size_t>(t) * n_q_heads + h) * D + part * kOutCols;
    uint32_t v[kOutCols];
    if (n_iters > 0) {
      if constexpr (kOutCols == 32) tmem_ld32(tDQ + lane_base + part * kOutCols, v);
      else tmem_ld16(tDQ + lane_base + part * kOutCols, v);
      tmem_wait_ld();
    } else {
#pragma unroll
      for (int e = 0; e < kOutCols; ++e) v[e] = 0u;
    }
    if (valid) {
      uint4* dst = reinterpret_cast<uint4*>(dq + row_off);
#pragma unroll
      for (int e = 0; e < kOutCols / 8; ++e) {
        uint4 w;
        w.x = pack_bf16x2(__uint_as_float(v[8 * e + 0]) * scale, __uint_as_float(v[8 * e + 1]) * scale);
        w.y = pack_bf16x2(__uint_as_float(v[8 * e + 2]) * scale, __uint_as_float(v[8 * e + 3]) * scale);
        w.z = pack_bf16x2(__uint_as_float(v[8 * e + 4]) * scale, __uint_as_float(v[8 * e + 5]) * scale);
        w.w = pack_bf16x2(__uint_as_float(v[8 * e + 6]) * scale, __uint_as_float(v[8 * e + 7]) * scale);
        dst[e] = w;
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, 512);
}

}  // namespace sap
