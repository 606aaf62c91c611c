"""GPU parity on seeded random packings: random document lengths (with empty and one-token documents), a random
chunk count that divides N, random MHA / GQA head counts, d in {64, 128}; forward and backward against the fp64
oracle, every element, through the C ABI.  Sizes span several 128-row tiles with ragged tails."""
import numpy as np
import pytest
import torch

import paper_2606_30460_b200 as sap
from oracle import oracle
from paper_2606_30460_b200.workloads import custom_workload, make_qkv
from parity import check_close, check_lse, to_np

pytestmark = pytest.mark.gpu


def random_case(seed):
    rng = np.random.default_rng(1000 + seed)
    n_docs = int(rng.integers(1, 9))
    kinds = rng.integers(0, 5, size=n_docs)
    lens = [int({0: 0, 1: 1}.get(int(k), rng.integers(2, 700))) for k in kinds]
    if sum(lens) == 0:
        lens[0] = int(rng.integers(1, 300))
    N = sum(lens)
    divisors = [p for p in range(1, 17) if N % p == 0]
    P = int(rng.choice(divisors))
    Hkv = int(rng.choice([1, 2, 3]))
    g = int(rng.choice([1, 2, 4]))
    d = int(rng.choice([64, 128]))
    return lens, P, Hkv * g, Hkv, d


@pytest.mark.parametrize("seed", range(16))
def test_random_packing_fwd_bwd(seed):
    lens, P, Hq, Hkv, d = random_case(seed)
    w = custom_workload(lens, P, Hq, Hkv, d, seed=seed, name=f"random{seed}")
    q, k, v, do = make_qkv(w, device="cpu")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    ref_plan = oracle.plan(w.cu_seqlens, w.n_chunks)
    assert plan.items.tobytes() == ref_plan.items.tobytes() and plan.kind_map.tobytes() == ref_plan.kind_map.tobytes()
    cu = plan.cu_seqlens_dev("cuda")
    qd, kd, vd, dod = q.cuda(), k.cuda(), v.cuda(), do.cuda()
    out, lse = sap.sap_attn_fwd(qd, kd, vd, cu, plan, softmax_scale=w.softmax_scale)
    dq = torch.full_like(qd, float("nan")); dk = torch.full_like(kd, float("nan")); dv = torch.full_like(vd, float("nan"))
    sap.sap_attn_bwd(dod, qd, kd, vd, out, lse, cu, plan, softmax_scale=w.softmax_scale, dq=dq, dk=dk, dv=dv)
    torch.cuda.synchronize()
    args = (to_np(q), to_np(k), to_np(v))
    tag = f"seed {seed} lens {lens} P {P} heads {Hq}/{Hkv} d {d}"
    o_ref, l_ref = oracle.attn_fwd(*args, w.cu_seqlens, w.softmax_scale)
    check_close(to_np(out), o_ref, f"{tag}: out")
    check_lse(to_np(lse).T, l_ref, f"{tag}: lse")
    check_close(to_np(dq), oracle.attn_bwd_dq(*args, to_np(do), w.cu_seqlens, w.softmax_scale), f"{tag}: dq")
    rdk, rdv = oracle.attn_bwd_dkv(*args, to_np(do), w.cu_seqlens, w.softmax_scale)
    check_close(to_np(dk), rdk, f"{tag}: dk")
    check_close(to_np(dv), rdv, f"{tag}: dv")


def test_split_and_fused_backward_agree():
    # the deterministic split form (7 GEMMs) and the fused form (5 GEMMs, atomic dQ) are two routes to one result
    w = custom_workload([700, 1100, 248 + 512], 5, 8, 2, 128)
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    fused = sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale)
    prev = sap.sap_debug_set_bwd_stages(7)
    try:
        split = sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale)
        split2 = sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale)
    finally:
        sap.sap_debug_set_bwd_stages(-1)
    torch.cuda.synchronize()
    assert prev == (1 | 8 | 16)
    for a, b, nm in zip(fused, split, ("dq", "dk", "dv")):
        check_close(to_np(a), to_np(b), f"fused vs split {nm}")
    for a, b in zip(split, split2):      # the split form is bit-reproducible
        assert torch.equal(a, b)


def test_three_backward_forms_agree_on_cfg2_full_size():
    """The library ships three routes to dQ / dK / dV: the CTA-pair kernel (default at head_dim 128), the one-CTA fused
    kernel (head_dim 64; sap_debug_set_bwd_form(1)) and the split, atomics-free form (sap_debug_set_bwd_stages(7), bit
    reproducible).  On configs[1] at full size - the launch configuration of the bench - all three agree within the
    tolerance and the split form repeats itself bit for bit; the default is checked against the oracle at this size in
    test_gpu_configs.py, so this ties the other two to it."""
    from paper_2606_30460_b200.workloads import make_workload
    w = make_workload(2)
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    run = lambda: sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale)
    pair = run()
    sap.sap_debug_set_bwd_form(1)
    try:
        one_cta = run()
    finally:
        sap.sap_debug_set_bwd_form(0)
    sap.sap_debug_set_bwd_stages(7)
    try:
        split, split2 = run(), run()
    finally:
        sap.sap_debug_set_bwd_stages(-1)
    torch.cuda.synchronize()
    for a, b, c, nm in zip(pair, one_cta, split, ("dq", "dk", "dv")):
        check_close(to_np(b), to_np(a), f"cfg2 one-CTA fused vs pair {nm}")
        check_close(to_np(c), to_np(a), f"cfg2 split vs pair {nm}")
    for a, b in zip(split, split2):
        assert torch.equal(a, b)
