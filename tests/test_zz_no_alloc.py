"""sap_attn_bwd_static: the backward pass for callers that cannot allocate device memory.

Some users of this library receive tensors but no allocator - a plug-in or callback inside a host framework whose memory
pool is the only thing allowed to allocate, or a process that has fixed its memory budget at start-up and may not call
cudaMalloc afterwards.  sap_attn_bwd is closed to them: it wants a workspace buffer, and its first call on a plan uploads
the plan with cudaMalloc.  sap_attn_bwd_static keeps the workspace and the plan's tile program in a fixed array built
into the library (16 MiB + 256 KiB per GPU) and so allocates nothing; larger problems are refused with status 10.

What is checked here, against the existing path (sap_attn_bwd with a caller workspace) on the same inputs:
dK and dV bit for bit (both paths run the same deterministic kernels), dQ within the tolerance of the other GPU tests
(tests/parity.py; its fp32 accumulation is atomic, so the last bits differ from run to run on either path) - on two calls
in a row with different data and different plans, because every call shares the one array and finds the previous call's
program, D and dQ sums in it.

The file is named so that pytest collects it last: with `pytest -x` a failure here cannot hide any other test.  It must
pass alone in a fresh process (then its first call is the library's first use of the device, and the plan has never
been uploaded) and after the other GPU tests.
"""
import pytest
import torch

import paper_2606_30460_b200 as sap
from paper_2606_30460_b200 import _lib
from paper_2606_30460_b200.workloads import custom_workload, make_qkv
from parity import check_close, to_np

pytestmark = pytest.mark.gpu


def both_paths(w, static_first):
    """Gradients of one workload from the no-allocation entry point and from sap_attn_bwd.  With `static_first` the
    no-allocation call runs before anything has uploaded this plan to the device."""
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    # the forward of a second plan over the same packing provides out / lse, so that `plan` itself stays un-uploaded
    fwd_plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    out, lse = sap.sap_attn_fwd(q, k, v, cu, fwd_plan, softmax_scale=w.softmax_scale)

    def static():
        g = [torch.full_like(t, float("nan")) for t in (q, k, v)]     # every element must be written
        sap.sap_attn_bwd_static(do, q, k, v, out, lse, cu, plan, *g, softmax_scale=w.softmax_scale)
        return g

    def existing():
        return list(sap.sap_attn_bwd(do, q, k, v, out, lse, cu, fwd_plan, softmax_scale=w.softmax_scale))

    if static_first:
        got = static()
        ref = existing()
    else:
        ref = existing()
        got = static()
    torch.cuda.synchronize()
    return got, ref


def compare(got, ref, what):
    (dq, dk, dv), (rdq, rdk, rdv) = got, ref
    assert torch.equal(dk, rdk), f"{what}: dk differs from sap_attn_bwd"
    assert torch.equal(dv, rdv), f"{what}: dv differs from sap_attn_bwd"
    check_close(to_np(dq), to_np(rdq), f"{what}: dq")


def test_two_calls_in_a_row_match_the_existing_path():
    # first call: GQA, head_dim 128 (the CTA-pair kernel), several pair-tiles and a ragged tail, 7.6 MiB of workspace
    a = custom_workload([700, 1100, 248 + 5], 1, 8, 2, 128, name="static_a")
    # second call: another packing, head count and head_dim (the one-CTA kernel), smaller than the first, so the array
    # still holds the first call's program and sums beyond what this call rewrites
    b = custom_workload([1, 300, 0, 33, 167, 64], 5, 4, 2, 64, name="static_b")
    ga, ra = both_paths(a, static_first=True)
    gb, rb = both_paths(b, static_first=False)
    compare(ga, ra, "first call")
    compare(gb, rb, "second call")
    # and the first problem once more, after the smaller one
    ga2, ra2 = both_paths(a, static_first=True)
    compare(ga2, ra2, "third call")


def test_sizes_beyond_the_built_in_scratch_are_refused():
    # 8192 tokens x 8 heads x 128: the workspace would be 32 MiB; the array holds 16
    w = custom_workload([8192], 1, 8, 2, 128, name="static_too_big")
    plan = sap.sap_plan(w.cu_seqlens, 1)
    assert sap.sap_workspace_bytes(plan, 8, 2, 128, sap.SAP_PASS_BWD) > 16 << 20
    q = torch.zeros(8192, 8, 128, dtype=torch.bfloat16, device="cuda")
    k = torch.zeros(8192, 2, 128, dtype=torch.bfloat16, device="cuda")
    lse = torch.zeros(8, 8192, dtype=torch.float32, device="cuda")
    with pytest.raises(sap.SapError) as e:
        sap.sap_attn_bwd_static(q, q, k, k, q, lse, plan.cu_seqlens_dev("cuda"), plan, torch.empty_like(q), torch.empty_like(k),
                                torch.empty_like(k))
    assert e.value.status == 10
    assert b"sap_attn_bwd_static" in _lib.lib().sap_strerror(10)
    # just inside the limit: 4096 tokens x 7 heads x 128 (14.1 MiB)
    plan_ok = sap.sap_plan([0, 4096], 1)
    assert sap.sap_workspace_bytes(plan_ok, 7, 7, 128, sap.SAP_PASS_BWD) <= 16 << 20
