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
