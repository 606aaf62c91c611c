"""GPU parity of the forward path (sap_attn_fwd, sap_attn_fwd_partial, sap_lse_merge) against the fp64
oracle, through the C ABI.  Tolerances: BASELINE.json north_star (max-abs 2e-2 / max-rel 1e-2 for bf16
out, 1e-3 absolute for fp32 LSE)."""
import numpy as np
import pytest
import torch

import paper_2606_30460_b200 as sap
from oracle import oracle
from paper_2606_30460_b200.workloads import custom_workload, make_qkv, make_workload
from parity import check_close, check_lse, to_np

pytestmark = pytest.mark.gpu


def run_fwd(w):
    q, k, v = make_qkv(w, device="cpu", with_dout=False)
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    before = sap.sap_launch_count()
    out, lse = sap.sap_attn_fwd(q.cuda(), k.cuda(), v.cuda(), cu, plan, softmax_scale=w.softmax_scale)
    torch.cuda.synchronize()
    assert sap.sap_launch_count() == before + 1
    return (q, k, v), plan, out, lse


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
}


@pytest.mark.parametrize("name", list(CASES))
def test_fwd_matches_oracle(name):
    lens, P, Hq, Hkv, d = CASES[name]
    w = custom_workload(lens, P, Hq, Hkv, d, name=name)
    (q, k, v), plan, out, lse = run_fwd(w)
    o_ref, l_ref = oracle.attn_fwd(to_np(q), to_np(k), to_np(v), w.cu_seqlens, w.softmax_scale)
    check_close(to_np(out), o_ref, f"{name}: out")
    check_lse(to_np(lse).T, l_ref, f"{name}: lse")


def test_fwd_cfg1_every_element():
    w = make_workload(1)
    (q, k, v), plan, out, lse = run_fwd(w)
    o_ref, l_ref = oracle.attn_fwd(to_np(q), to_np(k), to_np(v), w.cu_seqlens, w.softmax_scale)
    check_close(to_np(out), o_ref, "cfg1 out")
    check_lse(to_np(lse).T, l_ref, "cfg1 lse")


def test_fwd_q_zero_closed_form():
    # P6: Q = 0 => LSE_t = ln(t - s0 + 1), O_t = mean of v over [s0, t]
    w = custom_workload([200, 56, 300], 2, 2, 1, 64)
    q, k, v = make_qkv(w, device="cuda", with_dout=False)
    q.zero_()
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    out, lse = sap.sap_attn_fwd(q, k, v, plan.cu_seqlens_dev("cuda"), plan)
    cu = w.cu_seqlens
    pos = np.concatenate([np.arange(L) + 1 for L in w.doc_lens])
    check_lse(to_np(lse), np.broadcast_to(np.log(pos), (2, w.n_tokens)), "Q=0 lse")
    vf = to_np(v).astype(np.float64)
    ref = np.concatenate([np.cumsum(vf[cu[e]:cu[e + 1]], axis=0) / (np.arange(cu[e + 1] - cu[e]) + 1)[:, None, None]
                          for e in range(len(cu) - 1)])
    check_close(to_np(out), np.repeat(ref, 2, axis=1), "Q=0 out")


def test_fwd_poison_other_documents():
    # P8: huge K/V in every other document must not move this document's rows
    w = custom_workload([150, 300, 62], 4, 2, 2, 128)
    q, k, v = make_qkv(w, device="cuda", with_dout=False)
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    out0, lse0 = sap.sap_attn_fwd(q, k, v, cu, plan)
    k2, v2 = k.clone(), v.clone()
    k2[:150] = 60.0; v2[:150] = -1000.0; k2[450:] = 60.0; v2[450:] = 1000.0
    out1, lse1 = sap.sap_attn_fwd(q, k2, v2, cu, plan)
    assert torch.equal(out0[150:450], out1[150:450]) and torch.equal(lse0[:, 150:450], lse1[:, 150:450])


@pytest.mark.parametrize("d", [64, 128])
def test_partials_plus_merge_equal_fused(d):
    # P3 on the GPU path: per-item partials merged with sap_lse_merge == the fused forward == the oracle
    w = custom_workload([700, 1100, 248], 4, 4, 2, d)
    (q, k, v), plan, out, lse = run_fwd(w)
    qd, kd, vd = q.cuda(), k.cuda(), v.cuda()
    cu = plan.cu_seqlens_dev("cuda")
    N, Hq = w.n_tokens, w.n_q_heads
    acc_o = torch.zeros((N, Hq, d), dtype=torch.float32, device="cuda")
    acc_l = torch.full((Hq, N), float("-inf"), dtype=torch.float32, device="cuda")
    items = plan.items
    for it in range(plan.n_items):
        po, pl = sap.sap_attn_fwd_partial(qd, kd, vd, cu, plan, it, it + 1, softmax_scale=w.softmax_scale)
        # the partial of one item equals the oracle's partial for that item's rectangle
        qb, qe, kb, ke = (int(x) for x in items[it, 6:10])
        ro, rl = oracle.attn_partial(to_np(q), to_np(k), to_np(v), w.cu_seqlens, w.softmax_scale, qb, qe, kb, ke)
        got_l = to_np(pl).T[qb:qe]
        assert np.array_equal(np.isinf(got_l), np.isinf(rl))
        fin = np.isfinite(rl)
        assert np.abs(got_l[fin] - rl[fin]).max() <= 1e-3
        assert np.abs(to_np(po)[qb:qe] - ro).max() <= 2e-2
        outside = torch.ones(N, dtype=torch.bool, device="cuda"); outside[qb:qe] = False
        assert torch.isinf(pl[:, outside]).all() and (po[outside] == 0).all()
        acc_o, acc_l = sap.sap_lse_merge(acc_o, acc_l, po, pl, o_out=acc_o, lse_out=acc_l)
    o_ref, l_ref = oracle.attn_fwd(to_np(q), to_np(k), to_np(v), w.cu_seqlens, w.softmax_scale)
    check_close(to_np(acc_o), o_ref, "merged out")
    check_lse(to_np(acc_l).T, l_ref, "merged lse")
    check_close(to_np(acc_o), to_np(out), "merged vs fused")
    # bf16 output variant and row sub-range of the merge kernel
    half_o, half_l = sap.sap_lse_merge(acc_o, acc_l, torch.zeros_like(acc_o), torch.full_like(acc_l, float("-inf")),
                                       out_bf16=True, row_begin=100, row_end=1500)
    check_close(to_np(half_o)[100:1500], o_ref[100:1500], "merge with identity, bf16")
    assert (half_o[:100] == 0).all() and torch.isinf(half_l[:, 1500:]).all()


def test_merge_matches_oracle_random():
    g = torch.Generator().manual_seed(5)
    N, Hq, d = 300, 3, 64
    oa = torch.randn(N, Hq, d, generator=g); ob = torch.randn(N, Hq, d, generator=g)
    la = torch.randn(Hq, N, generator=g) * 5; lb = torch.randn(Hq, N, generator=g) * 5
    la[0, :10] = float("-inf"); lb[0, 5:15] = float("-inf")
    o, l = sap.sap_lse_merge(oa.cuda(), la.cuda(), ob.cuda(), lb.cuda())
    ro, rl = oracle.lse_merge(oa.numpy(), la.numpy().T, ob.numpy(), lb.numpy().T)
    got_l = to_np(l).T
    assert np.array_equal(np.isinf(got_l), np.isinf(rl))
    fin = np.isfinite(rl)
    assert np.abs(got_l[fin] - rl[fin]).max() < 1e-5
    both_inf = ~fin
    ro = np.where(both_inf[..., None], 0.0, ro)
    assert np.abs(to_np(o) - ro).max() < 1e-5


def test_fwd_rejects_bad_arguments():
    w = custom_workload([128], 1, 2, 1, 64)
    q, k, v = make_qkv(w, device="cuda", with_dout=False)
    plan = sap.sap_plan(w.cu_seqlens, 1)
    with pytest.raises(sap.SapError) as e:
        sap.sap_attn_fwd(q[:, :, :32].contiguous(), k[:, :, :32].contiguous(), v[:, :, :32].contiguous(),
                         plan.cu_seqlens_dev("cuda"), plan)
    assert e.value.status == 4


def test_fwd_persistent_scheduler_many_launches_two_streams():
    """The persistent forward takes its work items off {next, done} counter pairs that the last CTA of a launch re-arms
    (sap_api.cu: kSchedSlots = 4096 pairs per device and pool, handed out round-robin).  4400 launches - every pair of the
    eager pool reused - issued alternately on two streams, so launches overlap: every one must reproduce the first
    result bit for bit (the forward has no atomics on its outputs), with more work items than SMs and a ragged last
    tile.  A kernel that found its pair shared would trap and the final synchronize would raise."""
    w = custom_workload([3000, 1500, 2500 + 77, 1115], 4, 8, 2, 128, name="sched")
    q, k, v = (t.cuda() for t in make_qkv(w, device="cpu", with_dout=False))
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    ref_out, ref_lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = [[torch.empty_like(ref_out) for _ in range(3)] for _ in streams]
    lses = [[torch.empty_like(ref_lse) for _ in range(3)] for _ in streams]
    for it in range(2200):
        for si, st in enumerate(streams):
            o, l = outs[si][it % 3], lses[si][it % 3]
            sap.sap_attn_fwd(q, k, v, cu, plan, out=o, lse=l, softmax_scale=w.softmax_scale, stream=st)
    torch.cuda.synchronize()
    for si in range(2):
        for j in range(3):
            assert torch.equal(outs[si][j], ref_out), f"stream {si} buffer {j}: out differs"
            assert torch.equal(lses[si][j], ref_lse), f"stream {si} buffer {j}: lse differs"


def test_fwd_graph_replays_overlap_eager_launches():
    """A forward recorded into a CUDA graph keeps its counter pair for the life of the graph, so it must come from a
    pool that ordinary launches never draw from (sap.h, sap_attn_fwd): two graphs replayed on their own streams while a
    third stream issues ordinary launches - more of them than the eager pool has pairs, so an eager launch would have
    met a graph's pair had they shared a pool - must all reproduce the reference bit for bit."""
    w = custom_workload([3000, 1500, 2500 + 77, 1115], 4, 8, 2, 128, name="sched_graph")
    q, k, v = (t.cuda() for t in make_qkv(w, device="cpu", with_dout=False))
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    ref_out, ref_lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    torch.cuda.synchronize()
    graphs, g_out, g_lse, g_streams = [], [], [], []
    for _ in range(2):
        st = torch.cuda.Stream()
        st.wait_stream(torch.cuda.current_stream())
        o, l = torch.empty_like(ref_out), torch.empty_like(ref_lse)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(st):
            with torch.cuda.graph(g, stream=st):
                sap.sap_attn_fwd(q, k, v, cu, plan, out=o, lse=l, softmax_scale=w.softmax_scale)
        graphs.append(g); g_out.append(o); g_lse.append(l); g_streams.append(st)
    eager = torch.cuda.Stream()
    e_out = [torch.empty_like(ref_out) for _ in range(3)]
    e_lse = [torch.empty_like(ref_lse) for _ in range(3)]
    torch.cuda.synchronize()
    for it in range(4200):
        if it % 4 == 0:
            for g, st in zip(graphs, g_streams):
                with torch.cuda.stream(st):
                    g.replay()
        sap.sap_attn_fwd(q, k, v, cu, plan, out=e_out[it % 3], lse=e_lse[it % 3], softmax_scale=w.softmax_scale, stream=eager)
    torch.cuda.synchronize()
    for o, l in zip(g_out + e_out, g_lse + e_lse):
        assert torch.equal(o, ref_out) and torch.equal(l, ref_lse)


@pytest.mark.parametrize("name", list(CASES))
def test_fwd_row_pair_form_matches_oracle(name):
    """The row-pair form of the persistent forward (two 128-row halves of a 256-row tile of ONE q-head per work item: what
    sap_attn_fwd launches for odd Hq/Hkv, e.g. MHA, on long sequences) forced on every small case - one tile, ragged tails,
    empty and one-token documents, chunk lengths that are not multiples of 256, GQA and MHA, d = 64 and 128 - every element
    against the oracle."""
    lens, P, Hq, Hkv, d = CASES[name]
    w = custom_workload(lens, P, Hq, Hkv, d, name=name)
    prev = sap.sap_debug_set_fwd_form(2)
    try:
        (q, k, v), plan, out, lse = run_fwd(w)
    finally:
        sap.sap_debug_set_fwd_form(prev)
    o_ref, l_ref = oracle.attn_fwd(to_np(q), to_np(k), to_np(v), w.cu_seqlens, w.softmax_scale)
    check_close(to_np(out), o_ref, f"{name}: out (row pairs)")
    check_lse(to_np(lse).T, l_ref, f"{name}: lse (row pairs)")


def test_range_program_cache_eviction_two_streams_and_capture():
    """Range-restricted programs are cached per plan, 64 per kind, and an evicted one is freed only behind the last kernel
    that read it on EVERY stream (sap_api.cu: RangeUse).  136 one-item ranges - twice the cache - requested alternately on
    two streams, so programs built on one stream are evicted by calls on the other while their kernels are still queued:
    every partial must equal the one computed on a quiet device.  Then: the first use of a range inside stream capture
    is refused (building a program allocates and copies from pageable memory), a range seen before can be captured."""
    w = custom_workload([16 * 128], 16, 2, 2, 64, name="ranges")
    q, k, v = (t.cuda() for t in make_qkv(w, device="cpu", with_dout=False))
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    n = plan.n_items
    assert n == 136
    ref = []
    for it in range(n):
        ref.append(sap.sap_attn_fwd_partial(q, k, v, cu, plan, it, it + 1, softmax_scale=w.softmax_scale))
        torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    got = []
    for rep in range(2):
        for it in range(n):
            st = streams[(it + rep) % 2]
            with torch.cuda.stream(st):     # the result tensors are allocated on the stream that fills them
                got.append((it, sap.sap_attn_fwd_partial(q, k, v, cu, plan, it, it + 1, softmax_scale=w.softmax_scale, stream=st)))
    torch.cuda.synchronize()
    for it, (o, l) in got:
        assert torch.equal(o, ref[it][0]) and torch.equal(l, ref[it][1]), f"item {it}"
    # capture: item 0 was evicted long ago (miss), item n - 1 is in the cache (hit)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    o_g, l_g = torch.empty_like(ref[0][0]), torch.empty_like(ref[0][1])
    graph = torch.cuda.CUDAGraph()
    L = sap.api._lib.lib()
    args = lambda it: (q.data_ptr(), k.data_ptr(), v.data_ptr(), cu.data_ptr(), plan.handle, w.n_tokens, it, it + 1, o_g.data_ptr(),
                       l_g.data_ptr(), 2, 2, 64, float(w.softmax_scale), side.cuda_stream)
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            assert L.sap_attn_fwd_partial(*args(0)) == 4           # SAP_ERR_UNSUPPORTED, and the capture is still intact
            assert L.sap_attn_fwd_partial(*args(n - 1)) == 0
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(o_g, ref[n - 1][0]) and torch.equal(l_g, ref[n - 1][1])
