"""Stitched allocation (data plane; include/sap.h: sap_stitched_alloc) on ONE GPU: every [N, H, d]
tensor of the path lives in one virtual range made of P separately created physical allocations, one per sequence
chunk - the layout in which chunk c would be memory of the GPU that owns it.  The kernels (TMA loads through tensor
maps over the range, red.global into the dQ accumulator, plain stores) must not notice: the single launch and the P
per-rank launches on stitched tensors reproduce the run on ordinary allocations bit for bit (dQ: within tolerance, its
accumulation is atomic).  All chunks are on device 0 here: no second GPU exists on the box."""
import pytest
import torch

import paper_2606_30460_b200 as sap
from paper_2606_30460_b200.workloads import make_qkv, make_workload
from parity import check_close, to_np

pytestmark = pytest.mark.gpu


def stitched_like(t, P):
    """A tensor of t's shape and values inside a stitched range of P chunks along the token dimension."""
    n_rows = t.shape[0] // P
    chunk_bytes = n_rows * t[0].numel() * t.element_size()
    s = sap.Stitched(P, chunk_bytes)
    out = s.tensor(tuple(t.shape), t.dtype)
    out.copy_(t)
    return out


def test_granularity_and_errors():
    g = sap.Stitched.granularity(0)
    assert g >= 4096 and (g & (g - 1)) == 0
    s = sap.Stitched(3, g)
    assert s.nbytes == 3 * g and [s.owner(c) for c in range(4)] == [0, 0, 0, -1]
    x = s.tensor((3 * g,), torch.uint8)
    x.fill_(7)
    y = s.tensor((3 * g // 4,), torch.float32)                    # the chunks really are one contiguous range
    assert int(y.view(torch.uint8).sum().item()) == 7 * 3 * g
    del x, y
    s.free()
    with pytest.raises(sap.SapError) as e:                         # a chunk boundary must be an allocation boundary
        sap.Stitched(2, g + 512)
    assert e.value.status == 4


def test_fwd_bwd_on_stitched_tensors_cfg2():
    w = make_workload(2)                                           # 32K tokens, 8 chunks: 32 MiB (Q) / 8 MiB (K) per chunk
    P, Hq, Hkv, d = w.n_chunks, w.n_q_heads, w.n_kv_heads, w.head_dim
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, P)
    cu = plan.cu_seqlens_dev("cuda")
    ws = torch.empty(sap.sap_workspace_bytes(plan, Hq, Hkv, d, sap.SAP_PASS_BWD), dtype=torch.uint8, device="cuda")
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    dq, dk, dv = sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale, workspace=ws)
    torch.cuda.synchronize()

    sq, sk, sv, sdo = (stitched_like(t, P) for t in (q, k, v, do))
    nan = float("nan")
    so, sdq, sdk, sdv = (stitched_like(torch.full_like(t, nan), P) for t in (q, q, k, v))
    slse = torch.full_like(lse, nan)
    # one launch over the whole sequence
    sap.sap_attn_fwd(sq, sk, sv, cu, plan, out=so, lse=slse, softmax_scale=w.softmax_scale)
    sap.sap_attn_bwd(sdo, sq, sk, sv, so, slse, cu, plan, softmax_scale=w.softmax_scale, dq=sdq, dk=sdk, dv=sdv, workspace=ws)
    torch.cuda.synchronize()
    assert torch.equal(so, out) and torch.equal(slse, lse), "forward on stitched tensors differs"
    assert torch.equal(sdk, dk) and torch.equal(sdv, dv), "dK / dV on stitched tensors differ"
    check_close(to_np(sdq), to_np(dq), "dq, stitched vs ordinary allocation")

    # the P ranks' launches, each restricted to the chunk that would be its own memory
    for t in (so, sdq, sdk, sdv):
        t.fill_(nan)
    slse.fill_(nan)
    for c in range(P):
        sap.sap_attn_fwd_chunks(sq, sk, sv, cu, plan, c, c + 1, so, slse, softmax_scale=w.softmax_scale)
    for c in range(P):
        sap.sap_attn_bwd_begin(sdo, so, plan, c, c + 1, Hkv, ws)
    for c in reversed(range(P)):
        sap.sap_attn_bwd_chunks(sdo, sq, sk, sv, slse, cu, plan, c, c + 1, sdk, sdv, ws, softmax_scale=w.softmax_scale)
    for c in range(P):
        sap.sap_attn_bwd_end(plan, c, c + 1, sdq, Hkv, ws, softmax_scale=w.softmax_scale)
    torch.cuda.synchronize()
    assert torch.equal(so, out) and torch.equal(slse, lse), "per-rank forward on stitched tensors differs"
    assert torch.equal(sdk, dk) and torch.equal(sdv, dv), "per-rank dK / dV on stitched tensors differ"
    check_close(to_np(sdq), to_np(dq), "dq, per-rank launches on stitched tensors")


def test_rank_group_on_one_device_matches_oracle_and_single_launch():
    """ranks.RankGroup: the P ranks of one process, each launching on the chunk it owns, over stitched tensors, with the
    two group barriers of the backward - all chunks on device 0 (one stream: the launches run one after the other).
    Chunk = 8192 rows: 8 MiB of Q (4 heads of 128), 4 MiB of K / V (2 kv-heads)."""
    from oracle import oracle
    from paper_2606_30460_b200.ranks import RankGroup
    from paper_2606_30460_b200.workloads import custom_workload
    from parity import check_lse
    w = custom_workload([9000, 5000, 2384 + 16384], 4, 4, 2, 128, name="rank_group")     # 32768 tokens, 4 chunks of 8192
    P, Hq, Hkv, d = w.n_chunks, w.n_q_heads, w.n_kv_heads, w.head_dim
    q, k, v, do = make_qkv(w, device="cuda")
    grp = RankGroup(w.cu_seqlens, P)
    sq, sdo, so, sdq = (grp.tensor((Hq, d), torch.bfloat16) for _ in range(4))
    sk, sv, sdk, sdv = (grp.tensor((Hkv, d), torch.bfloat16) for _ in range(4))
    slse = grp.shared((Hq, w.n_tokens), torch.float32)
    ws = grp.workspace(Hq, Hkv, d)
    for dst, src in ((sq, q), (sk, k), (sv, v), (sdo, do)):
        dst.copy_(src)
    for t in (so, sdq, sdk, sdv, slse):
        t.fill_(float("nan"))
    grp.forward(sq, sk, sv, so, slse, softmax_scale=w.softmax_scale)
    grp.backward(sdo, sq, sk, sv, so, slse, sdq, sdk, sdv, ws, softmax_scale=w.softmax_scale)
    torch.cuda.synchronize()
    plan = sap.sap_plan(w.cu_seqlens, P)
    cu = plan.cu_seqlens_dev("cuda")
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    dq, dk, dv = sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale)
    torch.cuda.synchronize()
    assert torch.equal(so, out) and torch.equal(slse, lse) and torch.equal(sdk, dk) and torch.equal(sdv, dv)
    check_close(to_np(sdq), to_np(dq), "dq, rank group vs single launch")
    # sampled rows against the oracle (the last rows of the 18768-token document see keys of three chunks)
    rows = [0, 8999, 9000, 13999, 14000, 20000, 32767]
    args = (to_np(q), to_np(k), to_np(v))
    o_ref, l_ref = oracle.attn_fwd(*args, w.cu_seqlens, w.softmax_scale, rows=rows)
    check_close(to_np(so)[rows], o_ref, "rank group out (sampled rows)")
    check_lse(to_np(slse).T[rows], l_ref, "rank group lse (sampled rows)")
    dq_ref = oracle.attn_bwd_dq(*args, to_np(do), w.cu_seqlens, w.softmax_scale, rows=rows)
    check_close(to_np(sdq)[rows], dq_ref, "rank group dq (sampled rows)")
