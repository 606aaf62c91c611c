"""compile (sap_plan_schedule + sap_plan_codegen) -> execute (executor.sap_execute_fwd) with real
ranks on CPU (gloo).  Code lists pass the oracle's legality checker (oracle.check_codes: operands present before
`computing`, transfers paired, every partial returned, nothing redundant - a checker, not a second generator);
replaying them - with the ORACLE as the compute callable, the schedule is what is under test - reproduces the
unchunked attention on every rank, for the plain ring and for the balanced schedule (helpers compute on the K/V
rank, Q travels there, the partial result travels back)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import paper_2606_30460_b200 as sap
from oracle import oracle

HQ, HKV, D = 2, 1, 16
LAYOUTS = {"cfg1": [700, 1100, 248], "one_doc": [2048], "short_then_long": [100, 1948]}


def cu_of(docs):
    return np.concatenate([[0], np.cumsum(docs)]).astype(np.int64).tolist()


@pytest.mark.parametrize("name", list(LAYOUTS))
@pytest.mark.parametrize("P", [2, 4, 8])
@pytest.mark.parametrize("policy", [0, 1])
def test_codes_are_legal_and_pair_up(name, P, policy):
    cu = cu_of(LAYOUTS[name])
    plan = sap.sap_plan(cu, P)
    slots, n_stages = plan.schedule(policy)
    sends, recvs, computed = set(), set(), []
    lists = [plan.codegen(slots, r) for r in range(P)]
    assert oracle.check_codes(cu, P, slots, lists) == [], (name, P, policy)
    for r in range(P):
        codes = lists[r]
        assert (np.diff(codes[:, 0]) >= 0).all() and codes[:, 0].min() >= -1 and codes[:, 0].max() <= n_stages
        for st, op, tensor, peer, item in codes.tolist():
            if op == sap.SAP_OP_SEND:
                sends.add((st, tensor, r, peer, item))
            elif op == sap.SAP_OP_RECV:
                recvs.add((st, tensor, peer, r, item))
            elif op == sap.SAP_OP_COMPUTING:
                computed.append(item)
                assert (r, st) == tuple(slots[item])
    assert sends == recvs                                   # every send has its receive at the same stage on the peer
    assert sorted(computed) == list(range(plan.n_items))    # every block computed exactly once
    if policy == 0:                                         # the plain ring moves K/V only
        assert all(t == sap.SAP_T_KV for _, t, _, _, _ in sends)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, docs, policy, out_q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2606_30460_b200 import executor
        cu = np.asarray(cu_of(docs), dtype=np.int32)
        N, n = int(cu[-1]), int(cu[-1]) // world
        g = torch.Generator().manual_seed(11)
        q = torch.randn(N, HQ, D, generator=g).bfloat16().float()
        k = torch.randn(N, HKV, D, generator=g).bfloat16().float()
        v = torch.randn(N, HKV, D, generator=g).bfloat16().float()
        scale = D ** -0.5
        plan = sap.sap_plan(cu.tolist(), world)
        slots, _ = plan.schedule(policy)
        lo, hi = rank * n, (rank + 1) * n

        def partial_fn(item, q_shard, k_shard, v_shard):        # rows of chunk i against keys of chunk j, oracle arithmetic
            it = plan.items[item]
            i, j = int(it[0]), int(it[1])
            qg = np.zeros((N, HQ, D), np.float32); qg[i * n:(i + 1) * n] = q_shard.numpy()
            kg = np.zeros((N, HKV, D), np.float32); kg[j * n:(j + 1) * n] = k_shard.numpy()
            vg = np.zeros((N, HKV, D), np.float32); vg[j * n:(j + 1) * n] = v_shard.numpy()
            qb, qe, kb, ke = (int(x) for x in it[6:10])
            po, pl = oracle.attn_partial(qg, kg, vg, cu, scale, qb, qe, kb, ke)
            o = np.zeros((n, HQ, D)); l = np.full((n, HQ), -np.inf)
            o[qb - i * n:qe - i * n] = po; l[qb - i * n:qe - i * n] = pl
            return o, l

        merge_fn = lambda oa, la, ob, lb: oracle.lse_merge(oa, la, ob, lb)
        pack_o = lambda o, l: torch.from_numpy(np.concatenate([o, l[..., None]], axis=-1))
        unpack_o = lambda t: (t.numpy()[..., :D].copy(), t.numpy()[..., D].copy())
        kv = torch.stack([k[lo:hi], v[lo:hi]]).contiguous()
        o, l = executor.sap_execute_fwd(q[lo:hi].contiguous(), kv, plan, slots, rank, partial_fn, merge_fn, pack_o,
                                        unpack_o, torch.zeros((n, HQ, D + 1), dtype=torch.float64))
        o_ref, l_ref = oracle.attn_fwd(q.numpy(), k.numpy(), v.numpy(), cu, scale, rows=list(range(lo, hi)))
        out_q.put((rank, float(np.abs(o - o_ref).max()), float(np.abs(l - l_ref).max())))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("docs,world,policy", [([700, 1100, 248], 4, 1), ([2048], 4, 1), ([700, 1100, 248], 4, 0),
                                               ([100, 1948], 2, 1)])
def test_replaying_the_codes_reproduces_attention(docs, world, policy):
    ctx = mp.get_context("spawn")
    out_q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, docs, policy, out_q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out_q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, eo, el in res:
        assert eo < 1e-12 and el < 1e-12, (rank, eo, el)


# ------------------------------------------------------------------------------------------------ backward pass
@pytest.mark.parametrize("name", list(LAYOUTS))
@pytest.mark.parametrize("P", [2, 4, 8])
@pytest.mark.parametrize("policy", [0, 1])
def test_bwd_codes_are_legal_and_pair_up(name, P, policy):
    cu = cu_of(LAYOUTS[name])
    plan = sap.sap_plan(cu, P)
    slots, n_stages = plan.schedule(policy)
    sends, recvs, computed = set(), set(), []
    lists = [plan.codegen(slots, r, backward=True) for r in range(P)]
    assert oracle.check_codes(cu, P, slots, lists, backward=True) == [], (name, P, policy)
    for r in range(P):
        codes = lists[r]
        for st, op, tensor, peer, item in codes.tolist():
            if op == sap.SAP_OP_SEND:
                sends.add((st, tensor, r, peer, item))
            elif op == sap.SAP_OP_RECV:
                recvs.add((st, tensor, peer, r, item))
            elif op == sap.SAP_OP_COMPUTING:
                computed.append(item)
    assert sends == recvs and sorted(computed) == list(range(plan.n_items))
    kinds = {t for _, t, _, _, _ in sends}
    assert kinds <= {sap.SAP_T_Q, sap.SAP_T_KV, sap.SAP_T_DO, sap.SAP_T_DQ, sap.SAP_T_DKV}
    if policy == 0:                                         # plain ring: K/V out, dK/dV contributions back
        assert kinds <= {sap.SAP_T_KV, sap.SAP_T_DKV}


def _bwd_inputs(docs):
    cu = np.asarray(cu_of(docs), dtype=np.int32)
    N = int(cu[-1])
    g = torch.Generator().manual_seed(13)
    q = torch.randn(N, HQ, D, generator=g).bfloat16().float().numpy()
    k = torch.randn(N, HKV, D, generator=g).bfloat16().float().numpy()
    v = torch.randn(N, HKV, D, generator=g).bfloat16().float().numpy()
    do = torch.randn(N, HQ, D, generator=g).bfloat16().float().numpy()
    scale = D ** -0.5
    o, lse = oracle.attn_fwd(q, k, v, cu, scale)
    dsum = (do.astype(np.float64) * o).sum(-1)
    return cu, q, k, v, do, scale, lse, dsum


@pytest.mark.parametrize("docs,P", [([700, 1100, 248], 4), ([2048], 8), ([100, 1948], 2)])
def test_item_backward_sums_to_full_backward(docs, P):
    # pin of oracle.attn_bwd_item: the contributions of all plan items add up to the plain per-document backward
    cu, q, k, v, do, scale, lse, dsum = _bwd_inputs(docs)
    N = int(cu[-1])
    pl = oracle.plan(cu, P)
    dq = np.zeros((N, HQ, D)); dk = np.zeros((N, HKV, D)); dv = np.zeros((N, HKV, D))
    for it in pl.items:
        qb, qe, kb, ke = (int(x) for x in it[6:10])
        a, b, c = oracle.attn_bwd_item(q, k, v, do, lse, dsum, cu, scale, qb, qe, kb, ke)
        dq[qb:qe] += a; dk[kb:ke] += b; dv[kb:ke] += c
    assert np.abs(dq - oracle.attn_bwd_dq(q, k, v, do, cu, scale)).max() < 1e-10
    rdk, rdv = oracle.attn_bwd_dkv(q, k, v, do, cu, scale)
    assert np.abs(dk - rdk).max() < 1e-10 and np.abs(dv - rdv).max() < 1e-10


def _bwd_worker(rank, world, port, docs, policy, out_q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2606_30460_b200 import executor
        cu, q, k, v, do, scale, lse, dsum = _bwd_inputs(docs)
        N, n = int(cu[-1]), int(cu[-1]) // world
        plan = sap.sap_plan(cu.tolist(), world)
        slots, _ = plan.schedule(policy)
        lo, hi = rank * n, (rank + 1) * n

        def bwd_fn(item, q_shard, do_pack, kv):              # oracle arithmetic on what travelled
            it = plan.items[item]
            i, j = int(it[0]), int(it[1])
            qg = np.zeros((N, HQ, D)); qg[i * n:(i + 1) * n] = q_shard.numpy()
            dog = np.zeros((N, HQ, D)); lg = np.zeros((N, HQ)); dg = np.zeros((N, HQ))
            pk = do_pack.numpy()
            dog[i * n:(i + 1) * n] = pk[..., :D]; lg[i * n:(i + 1) * n] = pk[..., D]; dg[i * n:(i + 1) * n] = pk[..., D + 1]
            kg = np.zeros((N, HKV, D)); vg = np.zeros((N, HKV, D))
            kg[j * n:(j + 1) * n] = kv[0].numpy(); vg[j * n:(j + 1) * n] = kv[1].numpy()
            qb, qe, kb, ke = (int(x) for x in it[6:10])
            a, b, c = oracle.attn_bwd_item(qg, kg, vg, dog, lg, dg, cu, scale, qb, qe, kb, ke)
            dq = np.zeros((n, HQ, D)); dkv = np.zeros((2, n, HKV, D))
            dq[qb - i * n:qe - i * n] = a
            dkv[0, kb - j * n:ke - j * n] = b; dkv[1, kb - j * n:ke - j * n] = c
            return torch.from_numpy(dq), torch.from_numpy(dkv)

        q_shard = torch.from_numpy(q[lo:hi].astype(np.float64))
        do_pack = torch.from_numpy(np.concatenate([do[lo:hi].astype(np.float64), lse[lo:hi, :, None], dsum[lo:hi, :, None]], -1))
        kv = torch.from_numpy(np.stack([k[lo:hi], v[lo:hi]]).astype(np.float64))
        dq, dkv = executor.sap_execute_bwd(q_shard, do_pack, kv, plan, slots, rank, bwd_fn)
        rdq = oracle.attn_bwd_dq(q, k, v, do, cu, scale, rows=list(range(lo, hi)))
        rdk, rdv = oracle.attn_bwd_dkv(q, k, v, do, cu, scale, cols=list(range(lo, hi)))
        out_q.put((rank, float(np.abs(dq.numpy() - rdq).max()), float(np.abs(dkv[0].numpy() - rdk).max()),
                   float(np.abs(dkv[1].numpy() - rdv).max())))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("docs,world,policy", [([700, 1100, 248], 4, 1), ([2048], 4, 1), ([700, 1100, 248], 4, 0)])
def test_replaying_the_backward_codes_reproduces_the_gradients(docs, world, policy):
    ctx = mp.get_context("spawn")
    out_q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_bwd_worker, args=(r, world, port, docs, policy, out_q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out_q.get(timeout=240) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, eq, ek, ev in res:
        assert eq < 1e-10 and ek < 1e-10 and ev < 1e-10, (rank, eq, ek, ev)
