"""SURVEY 8(f) NEXT-1, host side: the plan-driven K/V exchange with real ranks, on CPU (gloo, world_size 2 and 4).
Every rank owns one sequence chunk, receives exactly the K/V shards its plan items name, computes the partials with
the ORACLE (the CUDA kernels need a GPU per rank; this test is about the schedule) and merges them; the result
must equal the unchunked oracle attention of its rows."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

DOCS = [700, 1100, 248]          # cfg1's packing: 2 SKIP pairs at P = 4
HQ, HKV, D = 2, 1, 16


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _inputs():
    g = torch.Generator().manual_seed(7)
    N = sum(DOCS)
    q = torch.randn(N, HQ, D, generator=g).bfloat16().float()
    k = torch.randn(N, HKV, D, generator=g).bfloat16().float()
    v = torch.randn(N, HKV, D, generator=g).bfloat16().float()
    return q, k, v


def _worker(rank, world, port, out_q, sub=None):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    group = None
    if sub is not None:           # the SAP ring runs over a strict subgroup whose ranks are not the global ranks
        group = dist.new_group(sub)
        if rank not in sub:
            dist.barrier()        # stay until the ring is done: the members' connections run through this process group
            dist.destroy_process_group()
            return
        rank, world = dist.get_group_rank(group, rank), len(sub)
    try:
        import paper_2606_30460_b200 as sap
        from paper_2606_30460_b200 import ring
        from oracle import oracle
        cu = np.concatenate([[0], np.cumsum(DOCS)]).astype(np.int32)
        N, n = int(cu[-1]), int(cu[-1]) // world
        q, k, v = _inputs()
        scale = D ** -0.5
        plan = sap.sap_plan(cu.tolist(), world)
        lo, hi = rank * n, (rank + 1) * n
        received = []

        def partial_fn(item, k_shard, v_shard):
            it = plan.items[item]
            j = int(it[1])
            received.append(j)
            kg = np.zeros((N, HKV, D), np.float32); vg = np.zeros((N, HKV, D), np.float32)
            kg[j * n:(j + 1) * n] = k_shard.numpy(); vg[j * n:(j + 1) * n] = v_shard.numpy()
            qg = np.zeros((N, HQ, D), np.float32); qg[lo:hi] = q[lo:hi].numpy()     # this rank only has its own Q rows
            qb, qe, kb, ke = (int(x) for x in it[6:10])
            po, pl = oracle.attn_partial(qg, kg, vg, cu, scale, qb, qe, kb, ke)
            o = np.zeros((n, HQ, D)); l = np.full((n, HQ), -np.inf)
            o[qb - lo:qe - lo] = po; l[qb - lo:qe - lo] = pl
            return o, l

        def merge_fn(oa, la, ob, lb):
            return oracle.lse_merge(oa, la, ob, lb)

        kv = torch.stack([k[lo:hi], v[lo:hi]]).contiguous()
        o, l = ring.sap_ring_fwd(kv, plan, rank, partial_fn, merge_fn, group=group)
        o_ref, l_ref = oracle.attn_fwd(q.numpy(), k.numpy(), v.numpy(), cu, scale, rows=list(range(lo, hi)))
        want = sorted(int(plan.items[x, 1]) for x in range(int(plan.chunk_offsets[rank]), int(plan.chunk_offsets[rank + 1])))
        out_q.put((rank, float(np.abs(o - o_ref).max()), float(np.abs(l - l_ref).max()), sorted(received), want))
        if sub is not None:
            dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 4])
def test_ring_forward_matches_unchunked(world):
    ctx = mp.get_context("spawn")
    out_q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out_q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out_q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, eo, el, got, want in res:
        assert eo < 1e-12 and el < 1e-12, (rank, eo, el)
        assert got == want                      # exactly the shards the plan names: skipped pairs move no data


def test_ring_over_a_subgroup_with_non_identity_ranks():
    # world of 3, the ring over global ranks {0, 2}: group rank 1 is global rank 2 (HSAP's inter-group communicator)
    ctx = mp.get_context("spawn")
    out_q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 3, port, out_q, [2, 0])) for r in range(3)]
    for p in procs:
        p.start()
    res = sorted(out_q.get(timeout=180) for _ in range(2))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert [r[0] for r in res] == [0, 1]
    for rank, eo, el, got, want in res:
        assert eo < 1e-12 and el < 1e-12 and got == want


def test_schedule_skips_what_the_plan_skips():
    import paper_2606_30460_b200 as sap
    from paper_2606_30460_b200 import ring
    cu = np.concatenate([[0], np.cumsum(DOCS)])
    plan = sap.sap_plan(cu.tolist(), 4)
    sched = ring.schedule(plan)
    # items (1,0), (2,1), (3,2), (3,1); pairs (2,0), (3,0) are SKIP
    assert sched == [[(0, 1), (1, 2), (2, 3)], [(1, 3)], []]
    for step, pairs in enumerate(sched, start=1):
        for src, dst in pairs:
            assert ring.step_peers(plan, src, step)[0] == dst and ring.step_peers(plan, dst, step)[1] == src
    one = sap.sap_plan([0, 2048], 4)           # a single document: the full ring, P(P-1)/2 transfers
    assert sum(len(s) for s in ring.schedule(one)) == 6
