"""SURVEY 8(f) NEXT-2 / NEXT-3 on the GPU: the compiled schedule (sap_plan_schedule) and the jitted code lists
(sap_plan_codegen, sap_plan_codegen_bwd; Table 1) of ALL P ranks are replayed in one process on one
B200 by executor.LocalExecutor - fixed staging buffers, device copies as the transport, and every arithmetic step a
kernel behind the C ABI (sap_attn_fwd_items, sap_lse_merge, sap_attn_bwd_begin / _items / _end, sap_axpy) - for the
plain ring and for the balanced schedule.  out / LSE / dQ / dK / dV are compared with the fp64 oracle.

Also: the per-item launches themselves (contributions of all items sum to the one-launch backward) and sap_axpy."""
import numpy as np
import pytest
import torch

import paper_2606_30460_b200 as sap
from oracle import oracle
from paper_2606_30460_b200 import executor
from paper_2606_30460_b200.workloads import custom_workload, make_qkv, make_workload
from parity import check_close, check_lse, to_np

pytestmark = pytest.mark.gpu


def replay(w, policy):
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    slots, n_stages = plan.schedule(policy)
    ex = executor.LocalExecutor(plan, slots, w.n_q_heads, w.n_kv_heads, w.head_dim, q.device, softmax_scale=w.softmax_scale)
    n0 = sap.sap_launch_count()
    out, lse = ex.forward(q, k, v, cu)
    dq, dk, dv = ex.backward(do, q, k, v, out, lse, cu)
    torch.cuda.synchronize()
    assert sap.sap_launch_count() - n0 >= 2 * plan.n_items      # one forward and one backward kernel per `computing` code
    return (q, k, v, do), (out, lse, dq, dk, dv), ex, n_stages


@pytest.mark.parametrize("policy", [sap.SAP_SCHED_RING, sap.SAP_SCHED_BALANCED])
@pytest.mark.parametrize("case", ["cfg1_packing_gqa_d128", "one_doc_8_ranks"])
def test_replay_all_ranks_small(case, policy):
    lens, P, Hq, Hkv, d = {"cfg1_packing_gqa_d128": ([700, 1100, 248], 4, 4, 2, 128),
                           "one_doc_8_ranks": ([2048], 8, 2, 1, 128)}[case]
    w = custom_workload(lens, P, Hq, Hkv, d, name=case)
    (q, k, v, do), (out, lse, dq, dk, dv), ex, n_stages = replay(w, policy)
    args = (to_np(q), to_np(k), to_np(v))
    o_ref, l_ref = oracle.attn_fwd(*args, w.cu_seqlens, w.softmax_scale)
    check_close(to_np(out), o_ref, f"{case} policy {policy} out")
    check_lse(to_np(lse).T, l_ref, f"{case} policy {policy} lse")
    check_close(to_np(dq), oracle.attn_bwd_dq(*args, to_np(do), w.cu_seqlens, w.softmax_scale), f"{case} policy {policy} dq")
    rdk, rdv = oracle.attn_bwd_dkv(*args, to_np(do), w.cu_seqlens, w.softmax_scale)
    check_close(to_np(dk), rdk, f"{case} policy {policy} dk")
    check_close(to_np(dv), rdv, f"{case} policy {policy} dv")
    if policy == sap.SAP_SCHED_BALANCED and case == "one_doc_8_ranks":
        assert n_stages == 8 // 2 + 1                          # closed form for one document: floor(P/2) + 1 stages
        assert ex.staging_slots["q"] >= 1 and ex.staging_slots["o"] >= 1   # helpers exist: Q travels, partials come back


@pytest.mark.parametrize("policy", [sap.SAP_SCHED_RING, sap.SAP_SCHED_BALANCED])
def test_replay_runs_in_buffers_allocated_once(policy):
    """"fixed global buffer ... no memory jitter".  Everything a replay needs - staging slots, compute
    buffers, the slots results wait in for their SEND, running results, workspaces - is allocated by LocalExecutor's
    constructor: device memory in use is the same at the start of every stage and after the last one, and over a whole
    forward / backward the peak exceeds the starting level by exactly the tensors the call returns."""
    w = custom_workload([2048], 8, 2, 1, 128, name="fixed_buffers")      # one document over 8 ranks: helpers in both passes
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    slots, _ = plan.schedule(policy)
    ex = executor.LocalExecutor(plan, slots, w.n_q_heads, w.n_kv_heads, w.head_dim, q.device, softmax_scale=w.softmax_scale)
    out, lse = ex.forward(q, k, v, cu)                # first use: range programs are built and uploaded by the library
    dq, dk, dv = ex.backward(do, q, k, v, out, lse, cu)
    del dq, dk, dv
    torch.cuda.synchronize()
    nbytes = lambda *ts: sum(t.numel() * t.element_size() for t in ts)
    for call, returned in ((lambda: ex.forward(q, k, v, cu), nbytes(out, lse)),
                           (lambda: ex.backward(do, q, k, v, out, lse, cu), nbytes(q, k, v))):
        base = torch.cuda.memory_allocated()
        torch.cuda.reset_peak_memory_stats()
        res = call()
        torch.cuda.synchronize()
        assert len(ex.mem_marks) >= 3 and set(ex.mem_marks) == {base}, ex.mem_marks
        assert torch.cuda.max_memory_allocated() - base <= returned + 4096 * len(res), (torch.cuda.max_memory_allocated() - base, returned)
        del res


@pytest.mark.parametrize("policy", [sap.SAP_SCHED_RING, sap.SAP_SCHED_BALANCED])
def test_replay_all_ranks_cfg2_equals_single_launch(policy):
    # BASELINE.json configs[1] at full size: the replay must reproduce the one-launch path (itself checked against the
    # oracle in test_gpu_configs.py) - out / dK / dV up to the rounding of the extra bf16 contributions, LSE to 1e-3
    w = make_workload(2)
    (q, k, v, do), (out, lse, dq, dk, dv), ex, _ = replay(w, policy)
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    out1, lse1 = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    dq1, dk1, dv1 = sap.sap_attn_bwd(do, q, k, v, out1, lse1, cu, plan, softmax_scale=w.softmax_scale)
    torch.cuda.synchronize()
    assert float((lse - lse1).abs().max()) <= 1e-3
    for name, a, b in (("out", out, out1), ("dq", dq, dq1), ("dk", dk, dk1), ("dv", dv, dv1)):
        check_close(to_np(a), to_np(b).astype(np.float64), f"cfg2 policy {policy} replay vs one launch: {name}")
    # and a sample of rows against the oracle
    rows = np.unique(np.random.default_rng(5).integers(0, w.n_tokens, size=128))
    sel = [0, 1, 2, 3]
    o_ref, l_ref = oracle.attn_fwd(to_np(q[:, sel]), to_np(k[:, :1]), to_np(v[:, :1]), w.cu_seqlens, w.softmax_scale, rows=rows)
    rt = torch.from_numpy(rows).cuda()
    check_close(to_np(out[rt][:, sel]), o_ref, f"cfg2 policy {policy} replay out vs oracle")
    check_lse(to_np(lse[sel][:, rt]).T, l_ref, f"cfg2 policy {policy} replay lse vs oracle")


def test_item_contributions_sum_to_the_one_launch_backward():
    w = custom_workload([700, 1100, 248 + 512], 5, 8, 2, 128, name="items")
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    dq1, dk1, dv1 = sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale)
    ws = torch.empty(sap.sap_workspace_bytes(plan, w.n_q_heads, w.n_kv_heads, w.head_dim, sap.SAP_PASS_BWD), dtype=torch.uint8, device="cuda")
    sap.sap_attn_bwd_begin(do, out, plan, 0, w.n_chunks, w.n_kv_heads, ws)
    dk_tot = torch.zeros(k.shape, dtype=torch.float32, device="cuda"); dv_tot = torch.zeros_like(dk_tot)
    for x in range(plan.n_items):
        sk = torch.full_like(k, float("nan")); sv = torch.full_like(v, float("nan"))
        sap.sap_attn_bwd_items(do, q, k, v, lse, cu, plan, x, x + 1, sk, sv, ws, softmax_scale=w.softmax_scale)
        kb, ke = int(plan.items[x, 8]), int(plan.items[x, 9])
        assert bool(torch.isfinite(sk[kb:ke]).all()) and bool(torch.isfinite(sv[kb:ke]).all())
        sap.sap_axpy(dk_tot[kb:ke], sk[kb:ke]); sap.sap_axpy(dv_tot[kb:ke], sv[kb:ke])
    dq = torch.empty_like(q)
    sap.sap_attn_bwd_end(plan, 0, w.n_chunks, dq, w.n_kv_heads, ws, softmax_scale=w.softmax_scale)
    torch.cuda.synchronize()
    args = (to_np(q), to_np(k), to_np(v), to_np(do), w.cu_seqlens, w.softmax_scale)
    check_close(to_np(dq), oracle.attn_bwd_dq(*args), "items dq")
    rdk, rdv = oracle.attn_bwd_dkv(*args)
    check_close(to_np(dk_tot), rdk, "items dk"); check_close(to_np(dv_tot), rdv, "items dv")
    check_close(to_np(dq), to_np(dq1).astype(np.float64), "items dq vs one launch")


def test_axpy_all_dtype_pairs():
    g = torch.Generator(device="cuda").manual_seed(3)
    for ddt in (torch.float32, torch.bfloat16):
        for sdt in (torch.float32, torch.bfloat16):
            dst = torch.randn(4096 + 8, generator=g, device="cuda").to(ddt)
            src = torch.randn(4096 + 8, generator=g, device="cuda").to(sdt)
            want = (dst.float() + 0.5 * src.float()).to(ddt)
            got = sap.sap_axpy(dst.clone(), src, 0.5)
            assert torch.equal(got, want), (ddt, sdt)
            got0 = sap.sap_axpy(torch.full_like(dst, float("nan")), src, 2.0, accumulate=False)
            assert torch.equal(got0, (2.0 * src.float()).to(ddt)), (ddt, sdt)
