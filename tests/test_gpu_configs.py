"""GPU parity at BASELINE.json's full sizes (configs[1..4] = cfg2..cfg5), in the launch configuration bench.py
times (all heads, whole sequence, one sap_attn_fwd + one sap_attn_bwd through the C ABI), on sampled outputs
the fp64 oracle computes one by one (SURVEY 8c "coverage tiers"):

  * out, LSE, dQ  : row-local -> a fixed row set (first / last rows of documents, chunk boundaries +-1,
                    128-tile boundaries, seeded random rows) for a subset of KV groups, every element of those rows;
  * dK, dV (dense dO): every key column in the tail window of the longest documents and every column of some
                    short documents (a column needs the row statistics of every later row of its document, so
                    early columns of long documents cost O(L^2) on the CPU);
  * dK, dV (sparse dO): dO is zero except on a seeded set of live rows; then EVERY key column of the subset's
                    kv-heads is compared (cost |live| x L on the CPU) - this is what reaches the early columns
                    of long documents, all tiles and all pipeline iterations of the dK/dV kernel;
  * properties that hold at any size: partials + sap_lse_merge == fused forward (P3), every output finite.

Heads and documents are independent problems (pins P2, GQA reading A-4), so the oracle is run on a head subset.
Tolerance: BASELINE.json north_star (tests/parity.py).
"""
import numpy as np
import pytest
import torch

import paper_2606_30460_b200 as sap
from oracle import oracle
from paper_2606_30460_b200.workloads import make_d64_workload, make_qkv, make_workload
from parity import check_close, check_lse, to_np, row_scale, col_scale

pytestmark = pytest.mark.gpu

# cfg -> (kv-heads the oracle checks, random rows, live rows of the sparse-dO pass)
PLAN = {2: ((0, 3, 7), 512, 512), 3: ((1, 6), 384, 384), 4: ((5,), 256, 256), 5: ((2,), 256, 320)}


def sample_rows(w, n_random, rng):
    cu, n, N = w.cu_seqlens, w.n_tokens // w.n_chunks, w.n_tokens
    rows = set()
    docs = sorted(range(len(w.doc_lens)), key=lambda e: -w.doc_lens[e])
    for e in docs[:12] + docs[-4:]:
        if w.doc_lens[e] > 0:
            rows.update((cu[e], min(cu[e] + 1, cu[e + 1] - 1), cu[e + 1] - 1))
    for i in range(1, w.n_chunks):          # chunk boundaries +-1 (ring-step edges)
        rows.update((i * n - 1, i * n, min(i * n + 1, N - 1)))
    for t in rng.integers(0, N // 128, size=16):  # 128-tile boundaries
        rows.update((int(t) * 128, min(int(t) * 128 + 127, N - 1)))
    rows.update(int(t) for t in rng.integers(0, N, size=n_random))
    return np.array(sorted(rows), dtype=np.int64)


def sample_cols(w, rng):
    cu = w.cu_seqlens
    docs = sorted(range(len(w.doc_lens)), key=lambda e: -w.doc_lens[e])
    cols = set()
    for e in docs[:4]:                       # tail window of the longest documents
        cols.update(range(max(cu[e], cu[e + 1] - 96), cu[e + 1]))
    short = [e for e in docs if 0 < w.doc_lens[e] <= 768][:6]
    for e in short:                          # whole short documents
        cols.update(range(cu[e], cu[e + 1]))
    return np.array(sorted(cols), dtype=np.int64)


@pytest.mark.parametrize("cfg", [2, 3, 4, 5])
def test_full_size_config_sampled_against_oracle(cfg):
    kv_sel, n_random, n_live = PLAN[cfg]
    check_full_size(make_workload(cfg), cfg, kv_sel, n_random, n_live, 100 + cfg)


def test_d64_context_workload_sampled_against_oracle():
    """head_dim 64 at the size bench.py reports it (`d64_context`: configs[2]'s 128K packing, 64 q-heads on 16 kv-heads):
    the persistent pair forward at d = 64 and sap_bwd_fused_kernel<64> over documents of up to ~1000 streamed tiles per
    row, where the small d = 64 cases stop at 9.  Same sampling as the configs above."""
    w = make_d64_workload()
    assert (w.n_tokens, w.n_q_heads, w.n_kv_heads, w.head_dim) == (131072, 64, 16, 64)
    check_full_size(w, "d64", (3, 11), 384, 384, 164)


def check_full_size(w, cfg, kv_sel, n_random, n_live, seed):
    N, Hq, Hkv, d = w.n_tokens, w.n_q_heads, w.n_kv_heads, w.head_dim
    g = Hq // Hkv
    q_sel = [hk * g + i for hk in kv_sel for i in range(g)]
    rng = np.random.default_rng(seed)
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    ref_plan = oracle.plan(w.cu_seqlens, w.n_chunks)
    assert plan.items.tobytes() == ref_plan.items.tobytes() and plan.kind_map.tobytes() == ref_plan.kind_map.tobytes()
    cu = plan.cu_seqlens_dev("cuda")
    n0 = sap.sap_launch_count()
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    dq = torch.full_like(q, float("nan")); dk = torch.full_like(k, float("nan")); dv = torch.full_like(v, float("nan"))
    sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale, dq=dq, dk=dk, dv=dv)
    torch.cuda.synchronize()
    assert sap.sap_launch_count() - n0 == 4      # the launch configuration bench.py times
    for name, t in (("out", out), ("lse", lse), ("dq", dq), ("dk", dk), ("dv", dv)):
        assert bool(torch.isfinite(t).all()), f"cfg{cfg} {name}: non-finite values"

    # the oracle's inputs: the same bf16 values, head subset, widened (float32 holds bf16 exactly)
    qs, dos = to_np(q[:, q_sel]), to_np(do[:, q_sel])
    ks, vs = to_np(k[:, list(kv_sel)]), to_np(v[:, list(kv_sel)])
    args = (qs, ks, vs)

    rows = sample_rows(w, n_random, rng)
    o_ref, l_ref = oracle.attn_fwd(*args, w.cu_seqlens, w.softmax_scale, rows=rows)
    rows_t = torch.from_numpy(rows).cuda()
    nk = row_scale(w.cu_seqlens, rows)
    check_close(to_np(out[rows_t][:, q_sel]), o_ref, f"cfg{cfg} out[{len(rows)} rows]", nk)
    check_lse(to_np(lse[q_sel][:, rows_t]).T, l_ref, f"cfg{cfg} lse")
    dq_ref = oracle.attn_bwd_dq(*args, dos, w.cu_seqlens, w.softmax_scale, rows=rows)
    check_close(to_np(dq[rows_t][:, q_sel]), dq_ref, f"cfg{cfg} dq[{len(rows)} rows]", nk)

    cols = sample_cols(w, rng)
    dk_ref, dv_ref = oracle.attn_bwd_dkv(*args, dos, w.cu_seqlens, w.softmax_scale, cols=cols)
    cols_t = torch.from_numpy(cols).cuda()
    nr = col_scale(w.cu_seqlens, cols)
    check_close(to_np(dk[cols_t][:, list(kv_sel)]), dk_ref, f"cfg{cfg} dk[{len(cols)} cols]", nr)
    check_close(to_np(dv[cols_t][:, list(kv_sel)]), dv_ref, f"cfg{cfg} dv[{len(cols)} cols]", nr)

    # sparse dO: every key column against the live rows
    live = np.unique(np.concatenate([rng.integers(0, N, size=n_live), rows[:: max(1, len(rows) // 48)]]))
    live_t = torch.from_numpy(live).cuda()
    do_sp = torch.zeros_like(do)
    do_sp[live_t] = do[live_t]
    dq2 = torch.full_like(q, float("nan")); dk2 = torch.full_like(k, float("nan")); dv2 = torch.full_like(v, float("nan"))
    sap.sap_attn_bwd(do_sp, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale, dq=dq2, dk=dk2, dv=dv2)
    torch.cuda.synchronize()
    dos_sp = to_np(do_sp[:, q_sel])
    dk_ref2, dv_ref2 = oracle.attn_bwd_dkv(*args, dos_sp, w.cu_seqlens, w.softmax_scale)
    check_close(to_np(dk2[:, list(kv_sel)]), dk_ref2, f"cfg{cfg} dk, sparse dO, all columns")
    check_close(to_np(dv2[:, list(kv_sel)]), dv_ref2, f"cfg{cfg} dv, sparse dO, all columns")
    dead = torch.ones(N, dtype=torch.bool, device="cuda"); dead[live_t] = False
    assert float(dq2[dead].abs().max()) == 0.0   # rows with dO = 0 have dQ = 0 exactly
    dq_ref2 = oracle.attn_bwd_dq(*args, dos_sp, w.cu_seqlens, w.softmax_scale, rows=live)
    check_close(to_np(dq2[live_t][:, q_sel]), dq_ref2, f"cfg{cfg} dq, sparse dO, live rows", row_scale(w.cu_seqlens, live))


def test_cfg2_partials_plus_merge_equal_fused_full_size():
    # P3 at full size: two disjoint item ranges, merged with sap_lse_merge, equal the fused forward
    w = make_workload(2)
    q, k, v = make_qkv(w, device="cuda", with_dout=False)
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    # split inside a q-chunk's item list so that rows really receive two partials
    co = plan.chunk_offsets
    multi = [i for i in range(w.n_chunks) if co[i + 1] - co[i] > 1]
    cut = int(co[multi[len(multi) // 2]] + 1) if multi else plan.n_items // 2
    oa, la = sap.sap_attn_fwd_partial(q, k, v, cu, plan, 0, cut, softmax_scale=w.softmax_scale)
    ob, lb = sap.sap_attn_fwd_partial(q, k, v, cu, plan, cut, plan.n_items, softmax_scale=w.softmax_scale)
    om, lm = sap.sap_lse_merge(oa, la, ob, lb, out_bf16=True)
    torch.cuda.synchronize()
    assert float((lm - lse).abs().max()) <= 1e-3
    diff = (om.float() - out.float()).abs()
    assert bool((diff <= torch.maximum(torch.tensor(2e-2, device="cuda"), 1e-2 * out.float().abs())).all())
