// sap_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, fp64 CPU oracle for the SAP attention hot path of
// "HSAP: A Hierarchical Sequence-aware Parallelism for Hybrid-Context
// Generative Models".  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference leg may call it.  It shares no code,
// header, table or helper with paper_2606_30460_b200/csrc (the CUDA path) and
// neither includes the other.
//
// What it computes and where the paper defines it:
//   * attention  Softmax(Q K^T / sqrt(d)) V                 PAPER.md:53-57 (sec 2.2.1, eq.)
//   * restricted to each packed segment ("cu_len ... only compute attention
//     within each segment"), causal                         PAPER.md:45 (sec 2.1)
//   * the method computes EXACT attention, so the float oracle is the
//     plain per-document definition, no tiling, no online softmax
//   * chunk-pair partial attention + "online" merge         PAPER.md:59, :239 (O-2), kept
//     separate so that "any chunking + merge == unchunked" can be tested as an invariant
//   * the plan: split of the mask over P contiguous equal chunks (PAPER.md:59 n=N/P,
//     :108 "Partition attention computation blocks"), brute definition
//
// Readings where the paper is silent: scale is an argument
// (A-1), key s visible to row t iff same document and s<=t (A-2), GQA q-head h uses
// kv-head h/(Hq/Hkv) (A-4), LSE is the natural log of the scaled scores (A-11),
// D uses the oracle's own fp64 O (A-12).
//
// Layouts: q,dout,O,dQ [N,Hq,d]; k,v,dK,dV [N,Hkv,d]; inputs are float32 arrays that
// hold the bf16 values exactly; everything is widened to double before any arithmetic.
// Parity status: every function below is pinned by tests/test_oracle_*.py (brute force
// full-matrix attention, per-document equivalence, chunk+merge invariance, finite
// differences, closed forms, printed plans under tests/golden/).  Nothing is unpinned.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// document containing token t: the unique e with cu[e] <= t < cu[e+1]   (A-9)
int doc_of(const int32_t* cu, int n_docs, int64_t t) {
  for (int e = 0; e < n_docs; ++e)
    if (cu[e] <= t && t < cu[e + 1]) return e;
  return -1;
}

struct Dims {
  int64_t N;
  int Hq, Hkv, d;
  double scale;
};

inline double dot(const float* a, const float* b, int d) {
  double acc = 0.0;
  for (int c = 0; c < d; ++c) acc += (double)a[c] * (double)b[c];
  return acc;
}

// One row of exact attention restricted to keys [lo, hi] (inclusive, already inside the
// row's document and <= t).  Returns lse (-inf if the key set is empty), fills o[d].
// scores: scratch of size >= hi-lo+1.
double attend_row(const Dims& D, const float* q, const float* k, const float* v, int64_t t, int h,
                  int64_t lo, int64_t hi, double* o, std::vector<double>& scores) {
  const int hk = h / (D.Hq / D.Hkv);
  for (int c = 0; c < D.d; ++c) o[c] = 0.0;
  if (hi < lo) return -std::numeric_limits<double>::infinity();
  const float* qt = q + (t * D.Hq + h) * D.d;
  const int64_t len = hi - lo + 1;
  if ((int64_t)scores.size() < len) scores.resize(len);
  double m = -std::numeric_limits<double>::infinity();
  for (int64_t s = lo; s <= hi; ++s) {
    const double x = D.scale * dot(qt, k + (s * D.Hkv + hk) * D.d, D.d);
    scores[s - lo] = x;
    m = std::max(m, x);
  }
  double sum = 0.0;
  for (int64_t i = 0; i < len; ++i) sum += std::exp(scores[i] - m);
  const double lse = m + std::log(sum);
  for (int64_t s = lo; s <= hi; ++s) {
    const double p = std::exp(scores[s - lo] - lse);
    const float* vs = v + (s * D.Hkv + hk) * D.d;
    for (int c = 0; c < D.d; ++c) o[c] += p * (double)vs[c];
  }
  return lse;
}

}  // namespace

extern "C" {

int sap_oracle_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// ---------------------------------------------------------------------------------
// O-1 forward.  For each listed row t (rows == nullptr: all N rows) and each q-head:
// O_t = sum_s P_ts v_s over s in [doc_start(t), t],  LSE_t = log sum_s exp(S_ts).
// out_o [n_rows,Hq,d] double, out_lse [n_rows,Hq] double.
// ---------------------------------------------------------------------------------
int sap_oracle_fwd(const float* q, const float* k, const float* v, const int32_t* cu, int n_docs,
                   int64_t N, int Hq, int Hkv, int d, double scale, const int64_t* rows,
                   int64_t n_rows, double* out_o, double* out_lse) {
  if (Hq % Hkv != 0 || cu[0] != 0 || cu[n_docs] != N) return 1;
  const Dims D{N, Hq, Hkv, d, scale};
  if (!rows) n_rows = N;
#pragma omp parallel
  {
    std::vector<double> scores;
#pragma omp for schedule(dynamic, 1) collapse(2)
    for (int64_t r = 0; r < n_rows; ++r)
      for (int h = 0; h < Hq; ++h) {
        const int64_t t = rows ? rows[r] : r;
        const int e = doc_of(cu, n_docs, t);
        out_lse[r * Hq + h] = attend_row(D, q, k, v, t, h, cu[e], t, out_o + (r * Hq + h) * d, scores);
      }
  }
  return 0;
}

// ---------------------------------------------------------------------------------
// Partial attention of one work item ("computing attention ... in an online
// manner"; Table 1 `computing`): rows [q_begin,q_end) against keys [kv_begin,kv_end),
// under the document AND causal mask.  Rows with no visible key get lse=-inf, o=0.
// out_o [(q_end-q_begin),Hq,d], out_lse [(q_end-q_begin),Hq].
// ---------------------------------------------------------------------------------
int sap_oracle_partial(const float* q, const float* k, const float* v, const int32_t* cu, int n_docs,
                       int64_t N, int Hq, int Hkv, int d, double scale, int64_t q_begin,
                       int64_t q_end, int64_t kv_begin, int64_t kv_end, double* out_o,
                       double* out_lse) {
  if (Hq % Hkv != 0) return 1;
  const Dims D{N, Hq, Hkv, d, scale};
#pragma omp parallel
  {
    std::vector<double> scores;
#pragma omp for schedule(dynamic, 1) collapse(2)
    for (int64_t t = q_begin; t < q_end; ++t)
      for (int h = 0; h < Hq; ++h) {
        const int e = doc_of(cu, n_docs, t);
        const int64_t lo = std::max<int64_t>(cu[e], kv_begin);
        const int64_t hi = std::min<int64_t>(t, kv_end - 1);
        const int64_t r = t - q_begin;
        out_lse[r * Hq + h] = attend_row(D, q, k, v, t, h, lo, hi, out_o + (r * Hq + h) * d, scores);
      }
  }
  return 0;
}

// ---------------------------------------------------------------------------------
// O-2 exact merge of two partials over disjoint key sets (online softmax, Milakov &
// Gimelshein, cited PAPER.md:59; "rescale" PAPER.md:239):
//   L = max(La,Lb) + log(exp(La-max) + exp(Lb-max)),  O = exp(La-L) Oa + exp(Lb-L) Ob,
// with (L=-inf, O=0) the identity and no NaN from (-inf) - (-inf).
// o_* [n,d], lse_* [n]; outputs may alias inputs a.
// ---------------------------------------------------------------------------------
int sap_oracle_merge(const double* o_a, const double* lse_a, const double* o_b, const double* lse_b,
                     int64_t n, int d, double* o_out, double* lse_out) {
  const double ninf = -std::numeric_limits<double>::infinity();
  for (int64_t i = 0; i < n; ++i) {
    const double la = lse_a[i], lb = lse_b[i];
    const double mx = std::max(la, lb);
    if (mx == ninf) {
      lse_out[i] = ninf;
      for (int c = 0; c < d; ++c) o_out[i * d + c] = 0.0;
      continue;
    }
    const double L = mx + std::log(std::exp(la - mx) + std::exp(lb - mx));
    const double wa = std::exp(la - L), wb = std::exp(lb - L);
    for (int c = 0; c < d; ++c) o_out[i * d + c] = wa * o_a[i * d + c] + wb * o_b[i * d + c];
    lse_out[i] = L;
  }
  return 0;
}

// ---------------------------------------------------------------------------------
// O-1 backward, dQ for listed rows (rows == nullptr: all).  With P_ts = exp(S_ts - LSE_t):
//   D_t = sum_c dO_tc O_tc;  dP_ts = sum_c dO_tc v_sc;  dS_ts = P_ts (dP_ts - D_t);
//   dQ_t = scale sum_s dS_ts k_s.                 out_dq [n_rows,Hq,d]
// (tensors dq/do exist in the paper's Table 1; fwd+bwd is what Table 2 times,:173)
// ---------------------------------------------------------------------------------
int sap_oracle_bwd_dq(const float* q, const float* k, const float* v, const float* dout,
                      const int32_t* cu, int n_docs, int64_t N, int Hq, int Hkv, int d, double scale,
                      const int64_t* rows, int64_t n_rows, double* out_dq) {
  if (Hq % Hkv != 0) return 1;
  const Dims D{N, Hq, Hkv, d, scale};
  if (!rows) n_rows = N;
#pragma omp parallel
  {
    std::vector<double> scores, o(d);
#pragma omp for schedule(dynamic, 1) collapse(2)
    for (int64_t r = 0; r < n_rows; ++r)
      for (int h = 0; h < Hq; ++h) {
        const int64_t t = rows ? rows[r] : r;
        const int hk = h / (Hq / Hkv);
        const int e = doc_of(cu, n_docs, t);
        const int64_t s0 = cu[e];
        const double lse = attend_row(D, q, k, v, t, h, s0, t, o.data(), scores);
        const float* dot_ = dout + (t * Hq + h) * d;
        const float* qt = q + (t * Hq + h) * d;
        double Dt = 0.0;
        for (int c = 0; c < d; ++c) Dt += (double)dot_[c] * o[c];
        double* dq = out_dq + (r * Hq + h) * d;
        for (int c = 0; c < d; ++c) dq[c] = 0.0;
        for (int64_t s = s0; s <= t; ++s) {
          const float* ks = k + (s * Hkv + hk) * d;
          const float* vs = v + (s * Hkv + hk) * d;
          const double p = std::exp(scale * dot(qt, ks, d) - lse);
          const double ds = p * (dot(dot_, vs, d) - Dt);
          for (int c = 0; c < d; ++c) dq[c] += scale * ds * (double)ks[c];
        }
      }
  }
  return 0;
}

// ---------------------------------------------------------------------------------
// O-1 backward, dK and dV for listed key positions (cols == nullptr: all):
//   dK_s = scale sum_{h in group} sum_{t>=s, same doc} dS_ts q_t
//   dV_s =       sum_{h in group} sum_{t>=s, same doc} P_ts dO_t
// Row statistics LSE_t, D_t are computed first (plain forward) for every row that some
// listed column can see.                      out_dk, out_dv [n_cols,Hkv,d]
// A row t whose dO_t is exactly zero in every head adds exactly zero to both sums
// (dP_ts = 0 and D_t = 0 give dS_ts = 0; P_ts dO_t = 0), so such rows are skipped: no value
// changes, and a test may probe all columns against a sparse set of live rows at full size.
// ---------------------------------------------------------------------------------
int sap_oracle_bwd_dkv(const float* q, const float* k, const float* v, const float* dout,
                       const int32_t* cu, int n_docs, int64_t N, int Hq, int Hkv, int d,
                       double scale, const int64_t* cols, int64_t n_cols, double* out_dk,
                       double* out_dv) {
  if (Hq % Hkv != 0) return 1;
  const Dims D{N, Hq, Hkv, d, scale};
  if (!cols) n_cols = N;
  const int g = Hq / Hkv;
  // rows whose statistics are needed: t >= (smallest listed column of t's document)
  std::vector<int64_t> first_col(n_docs, std::numeric_limits<int64_t>::max());
  for (int64_t i = 0; i < n_cols; ++i) {
    const int64_t s = cols ? cols[i] : i;
    const int e = doc_of(cu, n_docs, s);
    first_col[e] = std::min(first_col[e], s);
  }
  std::vector<char> live(N, 0);  // dO_t != 0 somewhere
  for (int64_t t = 0; t < N; ++t) {
    const float* row = dout + t * (int64_t)Hq * d;
    for (int64_t c = 0; c < (int64_t)Hq * d; ++c)
      if (row[c] != 0.0f) { live[t] = 1; break; }
  }
  std::vector<int64_t> need;
  for (int e = 0; e < n_docs; ++e)
    for (int64_t t = std::max<int64_t>(first_col[e], cu[e]); t < cu[e + 1]; ++t)
      if (live[t]) need.push_back(t);
  std::vector<int64_t> slot(N, -1);
  for (size_t i = 0; i < need.size(); ++i) slot[need[i]] = (int64_t)i;
  std::vector<double> lse(need.size() * Hq), Dt(need.size() * Hq);
#pragma omp parallel
  {
    std::vector<double> scores, o(d);
#pragma omp for schedule(dynamic, 1) collapse(2)
    for (int64_t i = 0; i < (int64_t)need.size(); ++i)
      for (int h = 0; h < Hq; ++h) {
        const int64_t t = need[i];
        const int e = doc_of(cu, n_docs, t);
        lse[i * Hq + h] = attend_row(D, q, k, v, t, h, cu[e], t, o.data(), scores);
        const float* dot_ = dout + (t * Hq + h) * d;
        double acc = 0.0;
        for (int c = 0; c < d; ++c) acc += (double)dot_[c] * o[c];
        Dt[i * Hq + h] = acc;
      }
  }
#pragma omp parallel for schedule(dynamic, 1) collapse(2)
  for (int64_t i = 0; i < n_cols; ++i)
    for (int hk = 0; hk < Hkv; ++hk) {
      const int64_t s = cols ? cols[i] : i;
      const int e = doc_of(cu, n_docs, s);
      const float* ks = k + (s * Hkv + hk) * d;
      const float* vs = v + (s * Hkv + hk) * d;
      double* dk = out_dk + (i * Hkv + hk) * d;
      double* dv = out_dv + (i * Hkv + hk) * d;
      for (int c = 0; c < d; ++c) dk[c] = dv[c] = 0.0;
      for (int64_t t = s; t < cu[e + 1]; ++t) {
        if (!live[t]) continue;  // contributes exactly zero
        for (int h = hk * g; h < (hk + 1) * g; ++h) {
          const float* qt = q + (t * Hq + h) * d;
          const float* dot_ = dout + (t * Hq + h) * d;
          const int64_t sl = slot[t];
          const double p = std::exp(scale * dot(qt, ks, d) - lse[sl * Hq + h]);
          const double ds = p * (dot(dot_, vs, d) - Dt[sl * Hq + h]);
          for (int c = 0; c < d; ++c) {
            dv[c] += p * (double)dot_[c];
            dk[c] += scale * ds * (double)qt[c];
          }
        }
      }
    }
  return 0;
}

// ---------------------------------------------------------------------------------
// O-3 plan, brute definition.  n = N/P, chunk c = tokens [c n, (c+1) n).
// For i in 0..P-1, for step s in 0..i, j = i-s (ring order, reading A-7): loop over ALL
// documents e; R = doc e ∩ chunk i, C = doc e ∩ chunk j; e contributes iff R, C non-empty
// and min(C) <= max(R).  No contributor -> SKIP (map only).  Else doc_lo/hi = min/max
// contributor, kind = DIAG if j==i else FULL, q range = hull of the R's, kv range = hull of
// the C's  ("partition the attention computation into local attention block").
// Item = 10 x int32: q_chunk, kv_chunk, doc_lo, doc_hi, mask_kind, step, q_begin, q_end,
// kv_begin, kv_end.  kind: 0 SKIP, 1 FULL, 2 DIAG.
// Outputs: items [<= P(P+1)/2][10], chunk_offsets [P+1] (CSR by q_chunk), kv_offsets [P+1] and
// kv_index [n_items] (CSR by kv_chunk, item indices ascending), kind_map [P*P] row-major.
// Returns n_items, or <0 on invalid input (-1 bad args, -2 bad cu_seqlens, -3 N % P != 0).
// ---------------------------------------------------------------------------------
int sap_oracle_plan(const int32_t* cu, int n_docs, int n_chunks, int32_t* items,
                    int32_t* chunk_offsets, int32_t* kv_offsets, int32_t* kv_index,
                    uint8_t* kind_map) {
  if (!cu || n_docs < 1 || n_chunks < 1) return -1;
  if (cu[0] != 0) return -2;
  for (int e = 0; e < n_docs; ++e)
    if (cu[e + 1] < cu[e]) return -2;
  const int64_t N = cu[n_docs];
  const int P = n_chunks;
  if (N <= 0 || N % P != 0) return -3;
  const int64_t n = N / P;
  std::memset(kind_map, 0, (size_t)P * P);
  int n_items = 0;
  for (int i = 0; i < P; ++i) {
    chunk_offsets[i] = n_items;
    for (int s = 0; s <= i; ++s) {
      const int j = i - s;
      int doc_lo = -1, doc_hi = -1;
      int64_t qb = N, qe = 0, kb = N, ke = 0;
      for (int e = 0; e < n_docs; ++e) {
        const int64_t r0 = std::max<int64_t>(cu[e], i * n), r1 = std::min<int64_t>(cu[e + 1], (i + 1) * n);
        const int64_t c0 = std::max<int64_t>(cu[e], j * n), c1 = std::min<int64_t>(cu[e + 1], (j + 1) * n);
        if (r0 >= r1 || c0 >= c1) continue;  // R or C empty
        if (c0 > r1 - 1) continue;           // min(C) > max(R): nothing causal
        if (doc_lo < 0) doc_lo = e;
        doc_hi = e;
        qb = std::min(qb, r0); qe = std::max(qe, r1);
        kb = std::min(kb, c0); ke = std::max(ke, c1);
      }
      if (doc_lo < 0) continue;
      const int kind = (j == i) ? 2 : 1;
      kind_map[(size_t)i * P + j] = (uint8_t)kind;
      int32_t* it = items + (size_t)n_items * 10;
      it[0] = i; it[1] = j; it[2] = doc_lo; it[3] = doc_hi; it[4] = kind; it[5] = s;
      it[6] = (int32_t)qb; it[7] = (int32_t)qe; it[8] = (int32_t)kb; it[9] = (int32_t)ke;
      ++n_items;
    }
  }
  chunk_offsets[P] = n_items;
  int pos = 0;
  for (int j = 0; j < P; ++j) {
    kv_offsets[j] = pos;
    for (int it = 0; it < n_items; ++it)
      if (items[(size_t)it * 10 + 1] == j) kv_index[pos++] = it;
  }
  kv_offsets[P] = pos;
  return n_items;
}

}  // extern "C"
