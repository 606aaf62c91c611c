"""Per-rank launches on ONE GPU: the P "ranks" run one after the other, each launching the
kernels restricted to its own chunks (sap_attn_fwd_chunks; sap_attn_bwd_begin / _chunks / _end).  No launch waits
on another.  Together they must reproduce the single launch: forward and dK / dV bit for bit (same tiles, same
order of accumulation), dQ within tolerance (its fp32 accumulation is atomic), and the oracle."""
import numpy as np
import pytest
import torch

import paper_2606_30460_b200 as sap
from oracle import oracle
from paper_2606_30460_b200.workloads import custom_workload, make_qkv, make_workload
from parity import check_close, check_lse, to_np

pytestmark = pytest.mark.gpu


def run_rank_by_rank(w, ranks_per_launch=1):
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    P, Hkv = w.n_chunks, w.n_kv_heads
    full_out, full_lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    full_dq, full_dk, full_dv = sap.sap_attn_bwd(do, q, k, v, full_out, full_lse, cu, plan, softmax_scale=w.softmax_scale)
    out = torch.full_like(q, float("nan")); lse = torch.full_like(full_lse, float("nan"))
    dq = torch.full_like(q, float("nan")); dk = torch.full_like(k, float("nan")); dv = torch.full_like(v, float("nan"))
    ws = torch.empty(sap.sap_workspace_bytes(plan, w.n_q_heads, Hkv, w.head_dim, sap.SAP_PASS_BWD), dtype=torch.uint8,
                     device="cuda")
    groups = [(a, min(a + ranks_per_launch, P)) for a in range(0, P, ranks_per_launch)]
    n0 = sap.sap_launch_count()
    for a, b in groups:                                             # every rank: its forward
        sap.sap_attn_fwd_chunks(q, k, v, cu, plan, a, b, out, lse, softmax_scale=w.softmax_scale)
    for a, b in groups:                                             # phase 1: D and a zeroed accumulator for own rows
        sap.sap_attn_bwd_begin(do, out, plan, a, b, Hkv, ws)
    for a, b in reversed(groups):                                   # phase 2 (any order): own K/V tiles
        sap.sap_attn_bwd_chunks(do, q, k, v, lse, cu, plan, a, b, dk, dv, ws, softmax_scale=w.softmax_scale)
    for a, b in groups:                                             # phase 3: own dQ rows
        sap.sap_attn_bwd_end(plan, a, b, dq, Hkv, ws, softmax_scale=w.softmax_scale)
    torch.cuda.synchronize()
    assert sap.sap_launch_count() - n0 == 4 * len(groups)
    return (q, k, v, do), (full_out, full_lse, full_dq, full_dk, full_dv), (out, lse, dq, dk, dv)


@pytest.mark.parametrize("lens,P,Hq,Hkv,d,rpl", [
    ([700, 1100, 248], 4, 4, 2, 128, 1),          # cfg1's packing with GQA: SKIP pairs, documents ending inside chunks
    ([2048], 8, 2, 2, 64, 1),                     # one document, MHA, d = 64: the one-head forward kernel
    ([300, 3000, 796], 16, 8, 2, 128, 3),         # several ranks per launch, ragged last group
])
def test_rank_by_rank_equals_single_launch_and_oracle(lens, P, Hq, Hkv, d, rpl):
    w = custom_workload(lens, P, Hq, Hkv, d)
    (q, k, v, do), full, part = run_rank_by_rank(w, rpl)
    for name, a, b in zip(("out", "lse", "dq", "dk", "dv"), part, full):
        assert bool(torch.isfinite(a).all()), f"{name}: rows left unwritten"
        if name == "dq":
            check_close(to_np(a), to_np(b), "dq rank by rank vs single launch")
        else:
            assert torch.equal(a, b), f"{name} differs from the single launch"
    args = (to_np(q), to_np(k), to_np(v))
    o_ref, l_ref = oracle.attn_fwd(*args, w.cu_seqlens, w.softmax_scale)
    check_close(to_np(part[0]), o_ref, "out"); check_lse(to_np(part[1]).T, l_ref, "lse")
    check_close(to_np(part[2]), oracle.attn_bwd_dq(*args, to_np(do), w.cu_seqlens, w.softmax_scale), "dq")


def test_rank_by_rank_cfg2_full_size():
    w = make_workload(2)
    _, full, part = run_rank_by_rank(w)
    for name, a, b in zip(("out", "lse", "dq", "dk", "dv"), part, full):
        if name == "dq":
            check_close(to_np(a), to_np(b), "cfg2 dq rank by rank vs single launch")
        else:
            assert torch.equal(a, b), f"cfg2 {name} differs from the single launch"


def test_chunk_api_rejects_bad_ranges_and_unaligned_chunks():
    w = custom_workload([300, 300], 3, 2, 2, 64)          # chunk_len 200: K/V tiles would straddle ranks
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, 3)
    cu = plan.cu_seqlens_dev("cuda")
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan)
    ws = torch.empty(sap.sap_workspace_bytes(plan, 2, 2, 64, sap.SAP_PASS_BWD), dtype=torch.uint8, device="cuda")
    with pytest.raises(sap.SapError) as e:
        sap.sap_attn_bwd_chunks(do, q, k, v, lse, cu, plan, 0, 1, torch.empty_like(k), torch.empty_like(v), ws)
    assert e.value.status == 4
    with pytest.raises(sap.SapError) as e:
        sap.sap_attn_fwd_chunks(q, k, v, cu, plan, 2, 5, out, lse)
    assert e.value.status == 1
    out2 = torch.full_like(out, float("nan")); lse2 = torch.full_like(lse, float("nan"))
    sap.sap_attn_fwd_chunks(q, k, v, cu, plan, 1, 2, out2, lse2)      # the forward has no alignment requirement
    torch.cuda.synchronize()
    assert torch.equal(out2[200:400], out[200:400]) and bool(torch.isnan(out2[:200]).all()) and bool(torch.isnan(out2[400:]).all())


@pytest.mark.parametrize("lens,P,Hq,Hkv,d", [
    ([2048], 8, 2, 2, 64),                        # MHA: chunks of 256 rows = one row-pair tile each
    ([700, 1100, 504], 6, 3, 1, 128),             # group of 3, chunks of 384 rows: a full pair tile and a half one per chunk
])
def test_rank_by_rank_forward_on_row_pairs(lens, P, Hq, Hkv, d):
    """The per-rank forward of odd Hq/Hkv in the row-pair form (forced: these shapes are below its size threshold): the P
    launches write only their own rows and together equal the oracle, every element."""
    w = custom_workload(lens, P, Hq, Hkv, d)
    q, k, v = make_qkv(w, device="cuda", with_dout=False)
    plan = sap.sap_plan(w.cu_seqlens, P)
    cu = plan.cu_seqlens_dev("cuda")
    out = torch.full_like(q, float("nan")); lse = torch.full((Hq, w.n_tokens), float("nan"), device="cuda")
    n = w.n_tokens // P
    prev = sap.sap_debug_set_fwd_form(2)
    try:
        for c in reversed(range(P)):
            sap.sap_attn_fwd_chunks(q, k, v, cu, plan, c, c + 1, out, lse, softmax_scale=w.softmax_scale)
            torch.cuda.synchronize()
            assert bool(torch.isnan(out[: c * n]).all()), "a rank wrote rows of an earlier chunk"
    finally:
        sap.sap_debug_set_fwd_form(prev)
    o_ref, l_ref = oracle.attn_fwd(to_np(q), to_np(k), to_np(v), w.cu_seqlens, w.softmax_scale)
    check_close(to_np(out), o_ref, "out, per-rank row pairs")
    check_lse(to_np(lse).T, l_ref, "lse, per-rank row pairs")
