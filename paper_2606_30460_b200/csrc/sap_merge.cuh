// Standalone exact LSE merge of two partial results over disjoint key sets
// (online softmax; the paper's separate "copy and rescale" operations, :239).
// HBM-bound elementwise kernel: 16-byte loads/stores.
#pragma once
#include <cuda_bf16.h>
#include <math_constants.h>
#include "sm100_ptx.cuh"

namespace sap {

constexpr int kMergeThreads = 256;

// A group of G lanes (G = head_dim/4 when that is a power of two <= 32, else 32) owns one (token, head)
// row: every lane reads both LSEs before any lane writes, so the outputs may alias the `a` inputs.
template <bool OUT_BF16>
__global__ void __launch_bounds__(kMergeThreads)
sap_lse_merge_kernel(const float* __restrict__ o_a, const float* __restrict__ lse_a, const float* __restrict__ o_b,
                     const float* __restrict__ lse_b, void* o_out, float* lse_out,
                     int64_t n_tokens, int n_q_heads, int head_dim, int64_t row_begin, int64_t n_rows, int group) {
  const int vec_per_row = head_dim / 4;  // float4 per (token, head)
  const int64_t gthread = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
  const int64_t groups_total = static_cast<int64_t>(gridDim.x) * blockDim.x / group;
  const int gl = static_cast<int>(gthread % group);
  const int64_t n_rows_pad = (n_rows + groups_total - 1) / groups_total * groups_total;  // warp-uniform trip count
  for (int64_t th = gthread / group; th < n_rows_pad; th += groups_total) {
    const bool live = th < n_rows;
    const int64_t t = row_begin + (live ? th : 0) / n_q_heads;
    const int h = static_cast<int>((live ? th : 0) % n_q_heads);
    const float la = lse_a[h * n_tokens + t], lb = lse_b[h * n_tokens + t];
    __syncwarp();
    const float m = fmaxf(la, lb);
    float wa = 0.f, wb = 0.f, l = -CUDART_INF_F;
    if (m > -CUDART_INF_F) {              // (-inf, 0) is the identity; no (-inf) - (-inf)
      const float ea = expf(la - m), eb = expf(lb - m);
      const float s = ea + eb;
      l = m + logf(s);
      wa = ea / s; wb = eb / s;
    }
    if (live) {
      for (int c = gl; c < vec_per_row; c += group) {
        const int64_t off = (t * n_q_heads + h) * head_dim + c * 4;
        const float4 a = *reinterpret_cast<const float4*>(o_a + off);
        const float4 b = *reinterpret_cast<const float4*>(o_b + off);
        float4 r;
        r.x = wa * a.x + wb * b.x; r.y = wa * a.y + wb * b.y; r.z = wa * a.z + wb * b.z; r.w = wa * a.w + wb * b.w;
        // a weight of exactly 0 must kill the term even when the dead side holds inf/nan
        if (wa == 0.f) r = make_float4(wb * b.x, wb * b.y, wb * b.z, wb * b.w);
        if (wb == 0.f) r = make_float4(wa * a.x, wa * a.y, wa * a.z, wa * a.w);
        if (wa == 0.f && wb == 0.f) r = make_float4(0.f, 0.f, 0.f, 0.f);
        if (OUT_BF16) {
          uint2 w;
          w.x = pack_bf16x2(r.x, r.y); w.y = pack_bf16x2(r.z, r.w);
          *reinterpret_cast<uint2*>(static_cast<__nv_bfloat16*>(o_out) + off) = w;
        } else {
          *reinterpret_cast<float4*>(static_cast<float*>(o_out) + off) = r;
        }
      }
      if (gl == 0) lse_out[h * n_tokens + t] = l;
    }
  }
}

}  // namespace sap
