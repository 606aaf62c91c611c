"""GPU parity of the backward path (sap_attn_bwd: D pre-pass, dK/dV kernel, dQ kernel) against the fp64
oracle, through the C ABI.  Tolerance: BASELINE.json north_star (max-abs 2e-2 / max-rel 1e-2 for bf16 grads)."""
import numpy as np
import pytest
import torch

import paper_2606_30460_b200 as sap
from oracle import oracle
from paper_2606_30460_b200.workloads import custom_workload, make_qkv, make_workload
from parity import check_close, to_np

pytestmark = pytest.mark.gpu


def run_bwd(w):
    q, k, v, do = make_qkv(w, device="cpu")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    qd, kd, vd, dod = q.cuda(), k.cuda(), v.cuda(), do.cuda()
    out, lse = sap.sap_attn_fwd(qd, kd, vd, cu, plan, softmax_scale=w.softmax_scale)
    # poison the outputs: every element must be written
    dq = torch.full_like(qd, float("nan")); dk = torch.full_like(kd, float("nan")); dv = torch.full_like(vd, float("nan"))
    before = sap.sap_launch_count()
    sap.sap_attn_bwd(dod, qd, kd, vd, out, lse, cu, plan, softmax_scale=w.softmax_scale, dq=dq, dk=dk, dv=dv)
    torch.cuda.synchronize()
    assert sap.sap_launch_count() == before + 3
    return (q, k, v, do), (dq, dk, dv)


CASES = {
    "one_tile_d128": ([128], 1, 1, 1, 128),
    "one_tile_d64": ([128], 1, 1, 1, 64),
    "one_token": ([1], 1, 1, 1, 64),
    "ragged_tail_d128": ([77, 130, 50], 1, 2, 1, 128),
    "many_short_docs": ([1, 2, 3, 1, 64, 5, 128, 129, 1, 50], 2, 4, 2, 64),
    "empty_docs": ([0, 100, 0, 0, 156, 0], 2, 2, 2, 128),
    "chunk_not_tile_multiple": ([300, 33, 167], 5, 4, 2, 64),
    "gqa_4_several_tiles": ([700, 1100, 248 + 512], 5, 8, 2, 128),
    "doc_starts_at_chunk_boundary": ([512, 512, 1024], 4, 2, 2, 64),
    "gqa_3_odd_group": ([300, 500, 96], 2, 6, 2, 128),
    "gqa_6_three_pairs": ([640, 384], 4, 6, 1, 64),
    "long_doc_many_iterations": ([1500, 548], 2, 4, 1, 128),
}


@pytest.mark.parametrize("name", list(CASES))
def test_bwd_matches_oracle(name):
    lens, P, Hq, Hkv, d = CASES[name]
    w = custom_workload(lens, P, Hq, Hkv, d, name=name)
    (q, k, v, do), (dq, dk, dv) = run_bwd(w)
    args = (to_np(q), to_np(k), to_np(v), to_np(do), w.cu_seqlens, w.softmax_scale)
    check_close(to_np(dq), oracle.attn_bwd_dq(*args), f"{name}: dq")
    rdk, rdv = oracle.attn_bwd_dkv(*args)
    check_close(to_np(dk), rdk, f"{name}: dk")
    check_close(to_np(dv), rdv, f"{name}: dv")


def test_bwd_cfg1_every_element():
    w = make_workload(1)
    (q, k, v, do), (dq, dk, dv) = run_bwd(w)
    args = (to_np(q), to_np(k), to_np(v), to_np(do), w.cu_seqlens, w.softmax_scale)
    check_close(to_np(dq), oracle.attn_bwd_dq(*args), "cfg1 dq")
    rdk, rdv = oracle.attn_bwd_dkv(*args)
    check_close(to_np(dk), rdk, "cfg1 dk")
    check_close(to_np(dv), rdv, "cfg1 dv")


def test_bwd_first_row_of_each_document():
    # P7: first row of a document sees only itself: dQ_t = 0; and a length-1 document gets dK = 0, dV = dO summed
    # over the q-heads of the group
    w = custom_workload([1, 130, 1, 124], 2, 4, 2, 64)
    (q, k, v, do), (dq, dk, dv) = run_bwd(w)
    for s0 in (0, 1, 131, 132):
        assert float(dq[s0].abs().max()) <= 1e-3   # P_tt (dP_tt - D_t) with D from the bf16-rounded O
    for s0 in (0, 131):
        assert float(dk[s0].abs().max()) <= 1e-3
        want = do[s0].float().view(2, 2, 64).sum(1)
        assert np.abs(to_np(dv[s0]) - want.numpy()).max() <= 2e-2


def test_bwd_independent_of_chunking():
    # P3 for gradients: any chunking gives the same result (within tolerance; accumulation order differs)
    lens = [700, 1100, 248]
    ref = None
    for P in (1, 2, 4, 8):
        w = custom_workload(lens, P, 4, 2, 64)
        _, grads = run_bwd(w)
        g = [to_np(x) for x in grads]
        if ref is None:
            ref = g
        else:
            for a, b, nm in zip(g, ref, ("dq", "dk", "dv")):
                check_close(a, b, f"P={P} {nm}")


def test_bwd_workspace_too_small():
    w = custom_workload([128], 1, 1, 1, 64)
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, 1)
    cu = plan.cu_seqlens_dev("cuda")
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan)
    with pytest.raises(sap.SapError) as e:
        sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))
    assert e.value.status == 5


def test_step_is_capturable_into_a_cuda_graph():
    """No attention call allocates, synchronises or reads device state on the host (sap.h: asynchronous on the caller's
    stream), so a whole step - forward, D pre-pass, accumulator zeroing, backward main kernel, dQ post pass - can be
    captured once and replayed: the replay must reproduce the eager results (forward, dK, dV bit for bit; dQ within
    tolerance: its accumulation is atomic).  The small, launch-bound shapes are where that pays."""
    w = custom_workload([700, 1100, 248], 4, 8, 2, 128, name="graph")
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    plan.upload()
    cu = plan.cu_seqlens_dev("cuda")
    ws = torch.empty(sap.sap_workspace_bytes(plan, w.n_q_heads, w.n_kv_heads, w.head_dim, sap.SAP_PASS_BWD), dtype=torch.uint8,
                     device="cuda")
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    dq, dk, dv = sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale, workspace=ws)
    torch.cuda.synchronize()
    g_out, g_lse = torch.empty_like(out), torch.empty_like(lse)
    g_dq, g_dk, g_dv = torch.empty_like(dq), torch.empty_like(dk), torch.empty_like(dv)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            sap.sap_attn_fwd(q, k, v, cu, plan, out=g_out, lse=g_lse, softmax_scale=w.softmax_scale)
            sap.sap_attn_bwd(do, q, k, v, g_out, g_lse, cu, plan, softmax_scale=w.softmax_scale, dq=g_dq, dk=g_dk, dv=g_dv,
                             workspace=ws)
    for rep in range(3):
        for t in (g_out, g_lse, g_dq, g_dk, g_dv):
            t.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(g_out, out) and torch.equal(g_lse, lse), f"replay {rep}: forward differs"
        assert torch.equal(g_dk, dk) and torch.equal(g_dv, dv), f"replay {rep}: dK / dV differ"
        check_close(to_np(g_dq), to_np(dq), f"replay {rep}: dq")
