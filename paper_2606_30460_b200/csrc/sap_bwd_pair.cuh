// Fused backward kernel on CTA pairs (head_dim 128): dK, dV and dQ from one pass over the visible
// (key tile, row tile) pairs, 5 GEMMs per pair, every MMA issued as tcgen05 cta_group::2.
// (Table 1 tensors do / dq / dkv; fwd+bwd is what the paper times, :173.)
//
// Why pairs: the one-CTA kernel (sap_bwd_fused.cuh) is bound by shared-memory bandwidth (128 B/clk per SM): an MMA with
// both operands in shared memory and N = 64 reads 6 KB per 32 tensor cycles.  A cluster of two CTAs on one TPC works on
// 256 keys (128 per CTA) x the same streamed 64-row Q/dO tile; each CTA then reads only HALF of every B operand (the
// hardware exchanges the halves), P^T and dS^T are A operands in TMEM, and the pair sums its two dQ^T partials inside
// the tensor core (K dimension = all 256 keys), which halves the fp32 reductions into the dQ accumulator.
//
// One cluster = one 256-row K/V pair-tile x one kv-head; CTA r of the pair owns keys [row0 + 128 r, row0 + 128 r + 128).
// 896 threads per CTA as in the one-CTA kernel: TMA warp, two issuer warps (only the leader CTA's issue; the peer's
// first one relays a barrier), one LSE/D loader warp, 16 compute warps, 8 drain warps.
// Per streamed 64-row tile of a q-head of the group (M = 256 = the pair's keys, 128 TMEM lanes per CTA):
//   S^T  = K Q^T, dP^T = V dO^T        A = own K / V tile [128 x d] (smem, K-major), B half = 32 of the 64 q rows
//   P^T  = 2^(scale*log2e*S^T - LSE),  dS^T = P^T (dP^T - D)        (compute warps; bf16 written back into TMEM)
//   dV  += P^T dO, dK += dS^T Q        A = P^T / dS^T (TMEM), B half = 64 of the 128 d columns of dO / Q (MN-major)
//   dQ^T = K^T dS^T  [128 (d) x 64 q]  M = 128: CTA r owns d in [64 r, 64 r + 64); A = K^T [64 d x 256 keys] (both key
//        tiles of the pair, its d half), B half = dS^T [256 keys x 32 q]: each CTA writes the dS^T rows of its own keys
//        into BOTH CTAs' buffers (its own q half locally, the other q half through distributed shared memory).
//   dQ^T is drained with red.global.add.f32 into dq_acc [N,Hq,d] (lane = d index: one 128-byte line per warp and row).
//
// TMEM (512 columns per CTA): [0,128) dK | [128,256) dV | two score buffers b at 256 + 128 b:
//   [0,64)   S^T fp32, free again as soon as the compute warps have read it; dQ^T of tile j then lands at [0,32) of buffer
//            (j+1)&1 (over S^T of tile j+1): lane = 64 (q / 32) + (d % 64), column = q % 32  (cta_group::2, M = 128 layout)
//   [64,128) dP^T fp32 -> per 16 q rows k: P^T bf16 at [64+16k, 64+16k+8), dS^T bf16 at [64+16k+8, 64+16k+16)
//            (the A operands of dV / dK: this region is the one with the long life, S^T(i+2) does not wait for it)
// Shared memory per CTA (224 KB): K 32 | V 32 | K^T 32 ([256 keys x own 64 d]) | Q 3 x 16 | dO 3 x 16 | dS^T 2 x 16.
//   A Q (dO) stage holds the four 32-row x 64-column boxes the CTA's B halves need, each at the same offset in both
//   CTAs because one descriptor addresses both: rows of q half r (both d halves) for S^T (dP^T), columns of d half r
//   (both q halves) for dK (dV).
#pragma once
#include <cuda_bf16.h>
#include <math_constants.h>
#include "sap_bwd_fused.cuh"

namespace sap {

constexpr int kPairKeys = 2 * kTile;   // keys of a pair-tile
constexpr int kPairThreads = kFusedThreads;
constexpr int kPairStages = 3;

struct PairSmem {  // head_dim 128 only
  static constexpr int D = 128;
  static constexpr int kKVBytes = kTile * D * 2;        // own K or V tile
  static constexpr int kKVBox = kTile * 128;            // [128 rows x 64 columns]
  static constexpr int kKTBytes = kPairKeys * 128;      // [256 keys x 64 d]
  static constexpr int kQSlot = 32 * 128;               // [32 rows x 64 columns]
  static constexpr int kQBytes = 4 * kQSlot;            // one Q or dO stage
  static constexpr int kDSBytes = kPairKeys * 64;       // dS^T [256 keys x 32 q], 64-byte rows
  static constexpr int kOffK = 0, kOffV = kKVBytes, kOffKT = 2 * kKVBytes, kOffQ = kOffKT + kKTBytes;
  static constexpr int kOffDO = kOffQ + kPairStages * kQBytes, kOffDS = kOffDO + kPairStages * kQBytes;
  static constexpr int kOffStat = kOffDS + 2 * kDSBytes;   // [stage][2][64] floats
  static constexpr int kBarOffset = kOffStat + kPairStages * 512;
  static constexpr int kTotal = kBarOffset + 512;
  static constexpr uint32_t kKVTxBytes = 2 * (2 * kKVBytes + kKTBytes);  // both CTAs: K, V, K^T
  static constexpr uint32_t kHalfTxBytes = 2 * 2 * 2 * kQSlot;           // both CTAs: two slots of Q and two of dO
};

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kPairThreads, 1)
sap_bwd_pair_kernel(const __grid_constant__ CUtensorMap mapQ32, const __grid_constant__ CUtensorMap mapDO32,
                    const __grid_constant__ CUtensorMap mapQ64, const __grid_constant__ CUtensorMap mapDO64,
                    const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV,
                    const TileDesc* __restrict__ tiles, const SegDesc* __restrict__ segs,
                    const int32_t* __restrict__ cu, int n_docs, const float* __restrict__ lse,
                    const float* __restrict__ dsum, float* __restrict__ dq_acc, __nv_bfloat16* __restrict__ dk,
                    __nv_bfloat16* __restrict__ dv, int n_tokens, int n_q_heads, int n_kv_heads, float scale,
                    float scale_log2) {
  using L = PairSmem;
  constexpr int D = 128;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = smem_raw;
  if (smem_u32(smem) & 1023u) __trap();
  const uint32_t s0 = smem_u32(smem);
  const uint32_t sK = s0 + L::kOffK, sV = s0 + L::kOffV, sKT = s0 + L::kOffKT, sQ = s0 + L::kOffQ, sDO = s0 + L::kOffDO,
                 sDS = s0 + L::kOffDS;
  float* stat = reinterpret_cast<float*>(smem + L::kOffStat);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::kBarOffset);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::kBarOffset + 496);
  // (L) = waited on in the leader CTA only, arrivals come from both CTAs; (B) = arrives in both CTAs by multicast commit
  // Q / dO stages are two rings: the q-half slots (B of S^T, dP^T), free again after dP^T; the d-half slots (B of dK, dV)
  const uint32_t bar_kv_full = smem_u32(bars + 0) /*L*/, bar_qs_full = smem_u32(bars + 1) /*L*/,
                 bar_qs_empty = smem_u32(bars + 4) /*B*/, bar_qm_full = smem_u32(bars + 28) /*L*/, bar_qm_empty = smem_u32(bars + 31) /*B*/, bar_stat_full = smem_u32(bars + 7),
                 bar_stat_empty = smem_u32(bars + 10), bar_s_full = smem_u32(bars + 13) /*B*/,
                 bar_p_full = smem_u32(bars + 15) /*L*/, bar_acc_full = smem_u32(bars + 17) /*B*/,
                 bar_dq_full = smem_u32(bars + 18) /*B*/, bar_dq_empty = smem_u32(bars + 20) /*L*/,
                 bar_ds_full = smem_u32(bars + 22) /*L: relay from the peer*/, bar_ds_land = smem_u32(bars + 24) /*own CTA*/,
                 bar_dpr = smem_u32(bars + 26) /*L*/, bar_dvk_done = smem_u32(bars + 34) /*leader: dV/dK(j) have read P^T, dS^T*/,
                 bar_p_full2 = smem_u32(bars + 36) /*L: second column part of every compute warp*/, bar_dpr2 = smem_u32(bars + 38) /*L: same for dpr*/;

  // logical warp id: service warps (0-3) are the physically last four (see sap_fwd.cuh)
  const int warp = ((threadIdx.x >> 5) + 4) % (kPairThreads / 32), lane = threadIdx.x & 31;
  const uint32_t cta = blockIdx.x & 1u;   // == %cluster_ctarank for cluster dims (2,1,1); written so that the compiler sees it is warp-uniform
  const int cid = blockIdx.x >> 1, n_tiles = (gridDim.x >> 1) / n_kv_heads;
  const int hk = cid / n_tiles, tile_idx = cid % n_tiles;
  const int g = n_q_heads / n_kv_heads;
  const TileDesc td = tiles[tile_idx];
  const int key0 = td.row0 + kTile * static_cast<int>(cta);  // first key of this CTA

  if (threadIdx.x == 0) {
    mbar_init(bar_kv_full, 1);
    for (int i = 0; i < kPairStages; ++i) {
      mbar_init(bar_qs_full + 8 * i, 1); mbar_init(bar_qs_empty + 8 * i, 1);
      mbar_init(bar_qm_full + 8 * i, 1); mbar_init(bar_qm_empty + 8 * i, 1);
      mbar_init(bar_stat_full + 8 * i, 32); mbar_init(bar_stat_empty + 8 * i, 2 * 4);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(bar_s_full + 8 * i, 1); mbar_init(bar_p_full + 8 * i, 2 * 4 * 2); mbar_init(bar_p_full2 + 8 * i, 2 * 4 * 2);
      mbar_init(bar_dq_full + 8 * i, 1); mbar_init(bar_dq_empty + 8 * i, 2 * 4 * kFusedDrainGroups);
      mbar_init(bar_ds_full + 8 * i, 1); mbar_init(bar_ds_land + 8 * i, 4); mbar_init(bar_dpr + 8 * i, 2 * 4 * 2); mbar_init(bar_dpr2 + 8 * i, 2 * 4 * 2);
      mbar_init(bar_dvk_done + 8 * i, 1);
    }
    mbar_init(bar_acc_full, 1);
    fence_mbar_init();
    tma_prefetch_desc(&mapQ32); tma_prefetch_desc(&mapDO32); tma_prefetch_desc(&mapQ64); tma_prefetch_desc(&mapDO64);
    tma_prefetch_desc(&mapK); tma_prefetch_desc(&mapV);
  }
  if (warp == 1) { tmem_alloc_pair(smem_u32(tmem_slot), 512); tmem_relinquish_pair(); }
  tc_fence_before();
  cluster_sync_all();   // barriers of both CTAs initialised before any remote arrive / TMA completion
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t tDK = tmem, tDV = tmem + 128, tBuf = tmem + 256;

  int iters_per_head = 0;
  for (int s = td.seg_begin; s < td.seg_end; ++s) iters_per_head += (segs[s].t_end - segs[s].t_begin + kBwdN - 1) / kBwdN;
  const int n_iters = iters_per_head * g;

  if (warp < 4) reg_dealloc<kFusedRegsService>();
  if (warp == 0) {
    // ------------------------------------------------------------------ TMA producer (each CTA loads its own operands)
    if (n_iters > 0 && elect_one()) {
      const uint32_t lead_kv_full = mapa_cluster(bar_kv_full, 0), lead_qs_full = mapa_cluster(bar_qs_full, 0),
                     lead_qm_full = mapa_cluster(bar_qm_full, 0);
      const int dcol = hk * D + 64 * static_cast<int>(cta);  // this CTA's d half
      if (cta == 0) mbar_expect_tx(bar_kv_full, L::kKVTxBytes);
      const uint64_t pol_once = l2_policy_evict_first();   // a pair's own K / V tiles are read by nobody else
#pragma unroll
      for (int b = 0; b < 2; ++b) {
        tma_load_2d_pair_hint(sK + b * L::kKVBox, &mapK, hk * D + b * 64, key0, lead_kv_full, pol_once);
        tma_load_2d_pair_hint(sV + b * L::kKVBox, &mapV, hk * D + b * 64, key0, lead_kv_full, pol_once);
        tma_load_2d_pair_hint(sKT + b * L::kKVBox, &mapK, dcol, td.row0 + b * kTile, lead_kv_full, pol_once);  // both key tiles, own d half
      }
      // the d-half slots of a tile are needed more than a tile later than its q-half slots: load them one tile behind,
      // so that waiting for their ring never holds back the next q-half loads
      int st = 0, ph = 1;  // empty barriers: the first pass over the ring must not block
      int pst = 0, pph = 1, ph_prev = -1, pt0 = 0;
      [[maybe_unused]] int tcount = 0;
      auto load_m = [&](int h, int t0, int stage, int phase) {
        mbar_wait(bar_qm_empty + 8 * stage, phase);
        if (cta == 0) mbar_expect_tx(bar_qm_full + 8 * stage, L::kHalfTxBytes);
        const uint32_t full = lead_qm_full + 8 * stage;
        const int qcol = h * D + 64 * static_cast<int>(cta);
        tma_load_2d_pair(sQ + stage * L::kQBytes + 2 * L::kQSlot, &mapQ64, qcol, t0, full);     // both q halves, d half r
        tma_load_2d_pair(sDO + stage * L::kQBytes + 2 * L::kQSlot, &mapDO64, qcol, t0, full);
      };
      for (int hq = 0; hq < g; ++hq) {
        const int h = hk * g + hq;
        for (int s = td.seg_begin; s < td.seg_end; ++s) {
          const int t_begin = segs[s].t_begin, t_end = segs[s].t_end;
          for (int t0 = t_begin; t0 < t_end; t0 += kBwdN) {
            mbar_wait(bar_qs_empty + 8 * st, ph);
            SAP_STAMP2(tcount, 10);
            if (cta == 0) mbar_expect_tx(bar_qs_full + 8 * st, L::kHalfTxBytes);
            const uint32_t full = lead_qs_full + 8 * st, q = sQ + st * L::kQBytes, o = sDO + st * L::kQBytes;
            const int tr = t0 + 32 * static_cast<int>(cta);  // this CTA's q half
            tma_load_2d_pair(q, &mapQ32, h * D, tr, full);                    // q half r, d half 0
            tma_load_2d_pair(q + L::kQSlot, &mapQ32, h * D + 64, tr, full);   // q half r, d half 1
            tma_load_2d_pair(o, &mapDO32, h * D, tr, full);
            tma_load_2d_pair(o + L::kQSlot, &mapDO32, h * D + 64, tr, full);
            SAP_STAMP2(tcount, 11);
            ++tcount;
            if (ph_prev >= 0) load_m(ph_prev, pt0, pst, pph);
            if (ph_prev >= 0 && ++pst == kPairStages) { pst = 0; pph ^= 1; }
            ph_prev = h; pt0 = t0;
            if (++st == kPairStages) { st = 0; ph ^= 1; }
          }
        }
      }
      if (ph_prev >= 0) load_m(ph_prev, pt0, pst, pph);
    }
  } else if (warp == 2) {
    // ------------------------------------------------------------------ per-row -LSE (log2 domain) and -D loader (negated: they are the addends of packed fma / add)
    int i = 0;
    for (int hq = 0; hq < g; ++hq) {
      const int h = hk * g + hq;
      const float* lse_h = lse + static_cast<size_t>(h) * n_tokens;
      const float* dsum_h = dsum + static_cast<size_t>(h) * n_tokens;
      for (int s = td.seg_begin; s < td.seg_end; ++s) {
        const int t_begin = segs[s].t_begin, t_end = segs[s].t_end;
        for (int t0 = t_begin; t0 < t_end; t0 += kBwdN, ++i) {
          const int st = i % kPairStages;
          float a[2], b[2];
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            const int t = t0 + lane + 32 * j;
            a[j] = t < n_tokens ? -__ldg(lse_h + t) * kLog2e : -CUDART_INF_F;
            b[j] = t < n_tokens ? -__ldg(dsum_h + t) : 0.f;
          }
          mbar_wait(bar_stat_empty + 8 * st, ((i / kPairStages) & 1) ^ 1);
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
    // ------------------------------------------------------------------ tcgen05 issuer (leader CTA, one elected thread)
    if (cta == 0 && n_iters > 0 && elect_one()) {
      constexpr uint32_t idesc_s = make_idesc_bf16(256, kBwdN, 0, 0);   // S^T, dP^T [256 x 64]: K-major x K-major
      const uint64_t dK0 = make_smem_desc(sK, 16, 1024), dV0 = make_smem_desc(sV, 16, 1024);
      const uint64_t dKT0 = make_smem_desc(sKT, L::kKVBox, 1024);                                   // K^T: MN-major A, M = own 64 d
      const uint64_t dQs0 = make_smem_desc(sQ, 16, 1024), dDOs0 = make_smem_desc(sDO, 16, 1024);    // K-major: q half r
      const uint64_t dQm0 = make_smem_desc(sQ + 2 * L::kQSlot, 2 * L::kQSlot, 1024);                // MN-major: d half r
      const uint64_t dDOm0 = make_smem_desc(sDO + 2 * L::kQSlot, 2 * L::kQSlot, 1024);
      const uint64_t dDS0 = make_smem_desc_sw(sDS, 4096, 512, kSwizzle64B);                         // dS^T: MN-major B, 32 q per CTA
      mbar_wait(bar_kv_full, 0);
      // Two issuing threads feed the one tensor pipe (it runs the MMAs in arrival order): this one S^T(i), dP^T(i); the
      // elected thread of warp 3 dQ^T(j), dV/dK(j).  Each waits only for its own inputs, so no cross-CTA hand-off of one
      // stream (200-600 cycles each) delays the other.  Every ordering between the streams is a barrier:
      //   S^T(i)  after S^T(i-2) was read and dQ^T(i-3) drained from these columns (dpr, dq_empty; both CTAs)
      //   dP^T(i) after dV/dK(i-2) have read P^T / dS^T from these columns        (dvk_done, committed by warp 3)
      for (int i = 0; i < n_iters; ++i) {
        const int b = i & 1, st = i % kPairStages;
        mbar_wait(bar_qs_full + 8 * st, (i / kPairStages) & 1);
        if (i >= 2) mbar_wait(bar_dpr2 + 8 * b, ((i - 2) >> 1) & 1);             // S^T(i-2) has been read from these columns (second parts last)
        if (i >= 3) mbar_wait(bar_dq_empty + 8 * (b ^ 1), ((i - 3) >> 1) & 1);   // ... and dQ^T(i-3), which followed it there, drained
        tc_fence_after();
        SAP_STAMP2(i, 18);
        const uint64_t dq = desc_add(dQs0, st * L::kQBytes), ddo = desc_add(dDOs0, st * L::kQBytes);
#pragma unroll
        for (int k = 0; k < D / 16; ++k)
          umma2_ss(tBuf + 128 * b, desc_add(dK0, (k / 4) * L::kKVBox + (k % 4) * 32), desc_add(dq, (k / 4) * L::kQSlot + (k % 4) * 32), idesc_s, k > 0);
        SAP_STAMP2(i, 0);
        if (i >= 2) { mbar_wait(bar_dvk_done + 8 * b, ((i - 2) >> 1) & 1); tc_fence_after(); }   // dV/dK(i-2) have read P^T, dS^T there
        SAP_STAMP2(i, 17);
#pragma unroll
        for (int k = 0; k < D / 16; ++k)
          umma2_ss(tBuf + 128 * b + 64, desc_add(dV0, (k / 4) * L::kKVBox + (k % 4) * 32), desc_add(ddo, (k / 4) * L::kQSlot + (k % 4) * 32), idesc_s, k > 0);
        umma2_commit(bar_s_full + 8 * b, 3);
        umma2_commit(bar_qs_empty + 8 * st, 3);   // the q-half slots of this stage are free once S^T(i), dP^T(i) are done
        SAP_STAMP2(i, 2);
      }
    } else if (cta == 1 && n_iters > 0 && elect_one()) {
      // relay: tell the leader when this CTA's dS^T buffer of tile j is complete (own rows stored, peer's rows landed)
      const uint32_t lead_ds_full = mapa_cluster(bar_ds_full, 0);
      for (int j = 0; j < n_iters; ++j) {
        mbar_wait(bar_ds_land + 8 * (j & 1), (j >> 1) & 1);
        fence_proxy_async_smem();
        mbar_arrive_cluster_relaxed(lead_ds_full + 8 * (j & 1));
      }
    }
  } else if (warp == 3) {
    // ------------------------------------------------------------------ second tcgen05 issuer (leader CTA): dQ^T(j-1), dV/dK(j)
    if (cta == 0 && n_iters > 0 && elect_one()) {
      constexpr uint32_t idesc_acc = make_idesc_bf16(256, D, 0, 1);     // dV, dK [256 x 128]: TMEM x MN-major
      constexpr uint32_t idesc_dq = make_idesc_bf16(128, kBwdN, 1, 1);  // dQ^T [128 x 64]: MN-major x MN-major
      const uint64_t dKT0 = make_smem_desc(sKT, L::kKVBox, 1024);                                   // K^T: MN-major A, M = own 64 d
      const uint64_t dQm0 = make_smem_desc(sQ + 2 * L::kQSlot, 2 * L::kQSlot, 1024);                // MN-major: d half r
      const uint64_t dDOm0 = make_smem_desc(sDO + 2 * L::kQSlot, 2 * L::kQSlot, 1024);
      const uint64_t dDS0 = make_smem_desc_sw(sDS, 4096, 512, kSwizzle64B);                         // dS^T: MN-major B, 32 q per CTA
      // Per tile j: dQ^T of tile j-1, then the dV / dK steps of tile j, those over the first column parts (q rows [0,32))
      // as soon as these are stored.  (dV / dK first halves ahead of dQ^T measured slower: 66.3 against 64.7 ms.)
      for (int j = 0; j <= n_iters; ++j) {
        const int bj = j & 1, stj = j % kPairStages;
        const uint32_t tPT = tBuf + 128 * bj + 64;
        const uint64_t dqm = desc_add(dQm0, stj * L::kQBytes), ddom = desc_add(dDOm0, stj * L::kQBytes);
        if (j >= 1) {
          const int q = j - 1, b = q & 1;   // dS^T buffer b; dQ^T goes to columns [0,32) of the S^T region of the other score buffer
          mbar_wait(bar_ds_land + 8 * b, (q >> 1) & 1);   // this CTA's dS^T buffer is complete
          mbar_wait(bar_ds_full + 8 * b, (q >> 1) & 1);   // ... and the peer's
          fence_proxy_async_smem();
          if (q + 1 < n_iters) mbar_wait(bar_dpr + 8 * (b ^ 1), ((q + 1) >> 1) & 1);               // columns [0,32) of S^T(q+1) (the first parts) have been read
          else if (q >= 2) mbar_wait(bar_dq_empty + 8 * b, ((q - 2) >> 1) & 1);                      // last tile: dQ^T(q-2) drained
          tc_fence_after();
          SAP_STAMP2(q, 12);
          const uint64_t dsb = desc_add(dDS0, b * L::kDSBytes);
#pragma unroll
          for (int k = 0; k < kPairKeys / 16; ++k)  // 16 keys per MMA
            umma2_ss(tBuf + 128 * (b ^ 1), desc_add(dKT0, k * 2048), desc_add(dsb, k * 1024), idesc_dq, k > 0);
          umma2_commit(bar_dq_full + 8 * b, 3);
          if (q == n_iters - 1) umma2_commit(bar_acc_full, 3);
          SAP_STAMP2(q, 4);
        }
        if (j < n_iters) {
          mbar_wait(bar_qm_full + 8 * stj, (j / kPairStages) & 1);
          mbar_wait(bar_p_full + 8 * bj, (j >> 1) & 1);
          tc_fence_after();
          SAP_STAMP2(j, 15);
#pragma unroll
          for (int k = 0; k < 2; ++k)   // k = 16 q rows = one column part
            umma2_ts(tDV, tPT + k * 16, desc_add(ddom, k * 2048), idesc_acc, (j > 0 || k > 0) ? 1u : 0u);
#pragma unroll
          for (int k = 0; k < 2; ++k)
            umma2_ts(tDK, tPT + k * 16 + 8, desc_add(dqm, k * 2048), idesc_acc, (j > 0 || k > 0) ? 1u : 0u);
          mbar_wait(bar_p_full2 + 8 * bj, (j >> 1) & 1);
          tc_fence_after();
#pragma unroll
          for (int k = 2; k < kBwdN / 16; ++k)
            umma2_ts(tDV, tPT + k * 16, desc_add(ddom, k * 2048), idesc_acc, 1u);
#pragma unroll
          for (int k = 2; k < kBwdN / 16; ++k)
            umma2_ts(tDK, tPT + k * 16 + 8, desc_add(dqm, k * 2048), idesc_acc, 1u);
          umma2_commit(bar_qm_empty + 8 * stj, 3);
          umma2_commit(bar_dvk_done + 8 * bj, 1);
          SAP_STAMP2(j, 3);
        }
      }
    }
  } else if (warp >= 4 + 4 * kFusedParts) {
    // ------------------------------------------------------------------ drain: dQ^T (TMEM) -> dq_acc (global, fp32 red)
    reg_dealloc<kFusedRegsDrain>();
    const int quarter = warp & 3, dpart = (warp - 4 - 4 * kFusedParts) >> 2;
    constexpr int kCols = 32 / kFusedDrainGroups;          // TMEM columns (q rows) per drain warp
    const int dcol = 64 * static_cast<int>(cta) + 32 * (quarter & 1) + lane;  // d index of this TMEM lane
    const int qoff = 16 * (2 * dpart + (quarter >> 1));                       // first q row of this warp's 16 columns: N half h = lane / 64 holds q rows [16 h, +16) and [32 + 16 h, +16)
    const uint32_t lane_base = static_cast<uint32_t>(quarter * 32) << 16;
    const size_t row_stride = static_cast<size_t>(n_q_heads) * D;
    const uint32_t lead_dq_empty = mapa_cluster(bar_dq_empty, 0);
    const uint64_t pol_acc = l2_policy_evict_last();   // accumulator lines: a miss is a DRAM read plus a write-back
    int j = 0;
    for (int hq = 0; hq < g; ++hq) {
      const int h = hk * g + hq;
      for (int s = td.seg_begin; s < td.seg_end; ++s) {
        const int t_begin = segs[s].t_begin, t_end = segs[s].t_end;
        for (int t0 = t_begin; t0 < t_end; t0 += kBwdN, ++j) {
          const int b = j & 1;
          const int tq = t0 + qoff;
          float* dst = dq_acc + (static_cast<size_t>(tq) * n_q_heads + h) * D + dcol;
          mbar_wait(bar_dq_full + 8 * b, (j >> 1) & 1);
          tc_fence_after();
          if (warp == 4 + 4 * kFusedParts && lane == 0) SAP_STAMP2(j, 8);
          uint32_t v[kCols];
          tmem_ld16(tBuf + 128 * (b ^ 1) + lane_base + kCols * dpart, v);
          tmem_wait_ld();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) { if (cta == 0) mbar_arrive(bar_dq_empty + 8 * b); else mbar_arrive_cluster_relaxed(lead_dq_empty + 8 * b); }  // these dQ^T columns are free again
          if (warp == 4 + 4 * kFusedParts && lane == 0) SAP_STAMP2(j, 9);
          if (tq + kCols <= n_tokens) {
#pragma unroll
            for (int c = 0; c < kCols; ++c) { red_add_f32_hint(dst, __uint_as_float(v[c]), pol_acc); dst += row_stride; }
          } else {
#pragma unroll
            for (int c = 0; c < kCols; ++c) {
              if (tq + c < n_tokens) red_add_f32_hint(dst, __uint_as_float(v[c]), pol_acc);
              dst += row_stride;
            }
          }
        }
      }
    }
  } else if (warp >= 4) {
    // ------------------------------------------------------------------ compute: P^T, dS^T; epilogue
    // Two groups of 8 warps take alternate tiles (group = tile parity = score buffer), so that one group's TMEM loads,
    // exponentials and stores overlap the other's; a warp covers one TMEM lane quarter (32 keys) x one q half (32 rows,
    // as two column parts of 16).
    reg_alloc<kFusedRegsCompute>();
    const int quarter = warp & 3, slot = (warp - 4) >> 2, group = slot & 1, qh = slot >> 1;
    const int r = quarter * 32 + lane;
    const int srow = key0 + r;                           // key index owned by this thread
    const bool valid = kTile * static_cast<int>(cta) + r < td.rows;
    const uint32_t lane_base = static_cast<uint32_t>(quarter * 32) << 16;
    const int32_t doc_hi = valid ? doc_end_of(cu, n_docs, srow) : 0;
    // dS^T row of this key in the [256 keys x 32 q] buffer of the CTA that owns q half qh: four 16-byte chunks,
    // 64-byte swizzle (chunk ^= bits 7-8 of the byte offset)
    const uint32_t prow = static_cast<uint32_t>(kTile * cta + r) * 64, psw = ((prow >> 7) & 3) << 4;
    const uint32_t ds_dst = mapa_cluster(sDS, static_cast<uint32_t>(qh));
    const uint32_t lead_p_full = mapa_cluster(bar_p_full, 0), lead_p_full2 = mapa_cluster(bar_p_full2, 0), lead_dpr = mapa_cluster(bar_dpr, 0), lead_dpr2 = mapa_cluster(bar_dpr2, 0);
    const uint32_t peer_ds_land = mapa_cluster(bar_ds_land, cta ^ 1);
    const bool ds_expect = quarter == 0;   // one of the 4 local-storing warps of a tile announces the peer's bytes
    uint8_t* const ds_local = (static_cast<uint32_t>(qh) == cta) ? smem + L::kOffDS : nullptr;  // own q half: plain stores
    const int b = group;
    const uint64_t scale2 = pack_f32x2(scale_log2, scale_log2);
    const uint32_t tS0 = tBuf + 128 * b + lane_base + kFusedCols * qh;

    int i = 0;
    for (int hq = 0; hq < g; ++hq) {
      for (int s = td.seg_begin; s < td.seg_end; ++s) {
        const SegDesc sd = segs[s];
        int lo = max(srow, sd.q_lo), hi = min(doc_hi, sd.q_hi);  // rows t that see key srow: [lo, hi)
        if (!valid || srow < sd.kv_lo || srow >= sd.kv_hi) { lo = 0; hi = 0; }
        for (int t0 = sd.t_begin; t0 < sd.t_end; t0 += kBwdN, ++i) {
          if ((i & 1) != group) continue;
          const int st = i % kPairStages;
          if (warp == 4 && lane == 0) SAP_STAMP2(i, 26);
          mbar_wait(bar_stat_full + 8 * st, (i / kPairStages) & 1);
          mbar_wait(bar_s_full + 8 * b, (i >> 1) & 1);
          tc_fence_after();
          if (warp == 4 && lane == 0) SAP_STAMP2(i, 5);
          uint32_t dsk[2][kFusedCols / 2];
#pragma unroll
          for (int pp = 0; pp < 2; ++pp) {
            const int part = 2 * pp + qh;   // first parts = q rows [0,32), second parts = [32,64): columns [0,32) of S^T are free for dQ^T early
            const uint32_t tST = tS0 + 2 * kFusedCols * pp, tDPT = tST + 64;
            const int tc = t0 + kFusedCols * part;  // first q row of this column part
            const bool need_mask = __any_sync(0xffffffffu, (tc < lo) || (tc + kFusedCols > hi));
            uint32_t sv[kFusedCols], dp[kFusedCols];
            tmem_ld16(tST, sv);
            tmem_ld16(tDPT, dp);
            const float4* l4 = reinterpret_cast<const float4*>(stat + st * 128 + kFusedCols * part);
            const float4* d4 = reinterpret_cast<const float4*>(stat + st * 128 + 64 + kFusedCols * part);
            tmem_wait_ld();
            if (warp == 4 && lane == 0 && pp == 0) SAP_STAMP2(i, 23);
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster_relaxed((pp ? lead_dpr2 : lead_dpr) + 8 * b);   // S^T and dP^T of this part are in registers: the S^T columns may take dQ^T(i-1).  (Both CTAs arrive through the cluster window: no branch on the CTA rank)
            if (lane == 0) { SAP_STAMP_MAX(i, 22); }
            if (need_mask) {  // boundary tiles only: masked scores become -inf, so P = 2^-inf = 0 and dS = 0
#pragma unroll
              for (int idx = 0; idx < kFusedCols; ++idx) {
                const int t = tc + idx;
                if (!(t >= lo && t < hi)) sv[idx] = 0xff800000u;
              }
            }
            uint32_t pk[kFusedCols];   // P^T (8 words) then dS^T (8 words): 16 TMEM columns
#pragma unroll
            for (int q4 = 0; q4 < kFusedCols / 4; ++q4) {
              const float4 lv = l4[q4], dvv = d4[q4];   // -LSE and -D of four q rows
              const uint64_t nl[2] = {pack_f32x2(lv.x, lv.y), pack_f32x2(lv.z, lv.w)};
              const uint64_t nd[2] = {pack_f32x2(dvv.x, dvv.y), pack_f32x2(dvv.z, dvv.w)};
#pragma unroll
              for (int e = 0; e < 2; ++e) {   // two q rows per packed instruction
                const int idx = q4 * 4 + 2 * e;
                float x0, x1;
                unpack_f32x2(fma_f32x2(pack_f32x2(__uint_as_float(sv[idx]), __uint_as_float(sv[idx + 1])), scale2, nl[e]), x0, x1);
                const float p0 = ex2_approx(x0), p1 = ex2_approx(x1);
                float s0, s1;
                unpack_f32x2(mul_f32x2(pack_f32x2(p0, p1), add_f32x2(pack_f32x2(__uint_as_float(dp[idx]), __uint_as_float(dp[idx + 1])), nd[e])), s0, s1);
                pk[q4 * 2 + e] = pack_bf16x2(p0, p1);
                pk[kFusedCols / 2 + q4 * 2 + e] = dsk[pp][q4 * 2 + e] = pack_bf16x2(s0, s1);
              }
            }
            if (warp == 4 && lane == 0 && pp == 0) SAP_STAMP2(i, 24);
            tmem_st16(tDPT, pk);  // bf16 P^T and dS^T over the 16 dP^T columns just read
            tmem_wait_st();
            if (warp == 4 && lane == 0 && pp == 0) SAP_STAMP2(i, 25);
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster_relaxed((pp ? lead_p_full2 : lead_p_full) + 8 * b);   // the dV / dK steps over these 16 q rows may start
            if (lane == 0) { SAP_STAMP_MAX(i, 20); SAP_STAMP_MIN(i, 21); }
          }
          if (i >= 2) mbar_wait(bar_dq_full + 8 * b, ((i >> 1) - 1) & 1);  // dQ^T of tile i-2 has read dS^T buffer b
          if (warp == 4 && lane == 0) SAP_STAMP2(i, 6);
          if (ds_local) {   // own q half: plain stores, counted as one arrival per warp on this CTA's barrier
            uint8_t* dsb = ds_local + b * L::kDSBytes;
#pragma unroll
            for (int c = 0; c < 4; ++c)
              *reinterpret_cast<uint4*>(dsb + ((prow + 16 * c) ^ psw)) = make_uint4(dsk[c >> 1][4 * (c & 1)], dsk[c >> 1][4 * (c & 1) + 1], dsk[c >> 1][4 * (c & 1) + 2], dsk[c >> 1][4 * (c & 1) + 3]);
            fence_proxy_async_smem();  // the dS^T stores must be visible to the tensor cores' (async proxy) reads
            __syncwarp();
            if (lane == 0) {
              if (ds_expect) mbar_expect_tx(bar_ds_land + 8 * b, kTile * 64);   // + the peer's 128 rows of 64 bytes (counts as this warp's arrival)
              else mbar_arrive(bar_ds_land + 8 * b);
            }
          } else {          // peer's q half: asynchronous stores, their bytes are counted on the peer's barrier
            const uint32_t dsb = ds_dst + b * L::kDSBytes, land = peer_ds_land + 8 * b;
#pragma unroll
            for (int c = 0; c < 4; ++c)
              st_async_v4(dsb + ((prow + 16 * c) ^ psw), dsk[c >> 1][4 * (c & 1)], dsk[c >> 1][4 * (c & 1) + 1], dsk[c >> 1][4 * (c & 1) + 2], dsk[c >> 1][4 * (c & 1) + 3], land);
            __syncwarp();
          }
          if (lane == 0) mbar_arrive(bar_stat_empty + 8 * st);
          if (warp == 4 && lane == 0) SAP_STAMP2(i, 7);
        }
      }
    }
    if (n_iters > 0) {
      mbar_wait(bar_acc_full, 0);
      tc_fence_after();
    }
    // parts 0,1 write the two column halves of dK (scaled), parts 2,3 those of dV
    const bool is_dk = slot < 2;
    const int chalf = slot & 1;
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
  cluster_sync_all();   // no CTA leaves (and frees its shared memory / TMEM) while the pair's MMAs or stores can touch it
  if (warp == 1) tmem_dealloc_pair(tmem, 512);
}

}  // namespace sap
