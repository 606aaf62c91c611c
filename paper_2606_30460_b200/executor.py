"""the "execute" half of SAP's compile-execute split - a rank replays
its jitted instruction list (sap_plan_codegen; Table 1 :85-98) stage by stage:

  * all SEND / RECV codes of a stage are posted as ONE batched isend/irecv (:124) and stay in flight while the
    stage's `computing` code runs (:122); the batch is waited for at the end of the stage;
  * COPY codes then move what arrived: q / kv into the compute buffers of the item they belong to, a partial result
    o into this rank's running (O, LSE) by the exact log-sum-exp merge ("copy and rescale", :239);
  * receive buffers are one shard each (the paper's fixed multiple of (N/P) x H x d, :140).

Forward pass.  The arithmetic is two callables, as in ring.py: `partial_fn(item, q_shard, k_shard, v_shard) ->
(o [n,Hq,d], lse)` over the rows of chunk q_chunk(item) and `merge_fn`; `ring.cuda_fns`-style adapters provide them
on a GPU, the CPU tests (gloo) inject the oracle's.  Not run on more than one GPU (this build has one).
"""
from __future__ import annotations

from typing import Callable

import numpy as np

from .api import (Plan, SAP_OP_COMPUTING, SAP_OP_COPY, SAP_OP_RECV, SAP_OP_SEND, SAP_T_DKV, SAP_T_DO, SAP_T_DQ, SAP_T_KV,
                  SAP_T_O, SAP_T_Q)


def sap_execute_fwd(q_shard, kv_shard, plan: Plan, slots: np.ndarray, rank: int, partial_fn: Callable,
                    merge_fn: Callable, pack_o: Callable, unpack_o: Callable, o_template, group=None):
    """Replays rank `rank`'s code list.  q_shard [n,Hq,d], kv_shard [2,n,Hkv,d]: this rank's tensors.  pack_o(o, lse)
    -> one tensor to send, unpack_o(tensor) -> (o, lse), o_template: a tensor shaped like pack_o's result (receive
    buffers are allocated like it).  Returns this rank's merged (o, lse) (None, None if the rank
    owns no rows with visible keys, which cannot happen: the diagonal item always exists)."""
    import torch
    import torch.distributed as dist

    codes = plan.codegen(slots, rank)
    items = plan.items
    stages = sorted(set(int(c[0]) for c in codes))
    q_buf, kv_buf, results, acc = {}, {}, {}, None           # per item: received q / kv; computed partials to send
    for st in stages:
        mine = [c for c in codes if int(c[0]) == st]
        ops, recv = [], {}
        for _, op, tensor, peer, item in (tuple(int(v) for v in c) for c in mine):
            if op == SAP_OP_SEND:
                payload = q_shard if tensor == SAP_T_Q else kv_shard if tensor == SAP_T_KV else pack_o(*results.pop(item))
                ops.append(dist.P2POp(dist.isend, payload.contiguous(), peer, group))
            elif op == SAP_OP_RECV:
                like = q_shard if tensor == SAP_T_Q else kv_shard if tensor == SAP_T_KV else o_template
                recv[(tensor, peer, item)] = torch.empty_like(like)
                ops.append(dist.P2POp(dist.irecv, recv[(tensor, peer, item)], peer, group))
        reqs = dist.batch_isend_irecv(ops) if ops else []      # one batch per stage, in flight during the computing code
        for _, op, tensor, peer, item in (tuple(int(v) for v in c) for c in mine):
            if op != SAP_OP_COMPUTING:
                continue
            i, j = int(items[item, 0]), int(items[item, 1])
            qs = q_shard if i == rank else q_buf.pop(item)
            kv = kv_shard if j == rank else kv_buf.pop(item)
            o, lse = partial_fn(item, qs, kv[0], kv[1])
            if i == rank:
                acc = (o, lse) if acc is None else merge_fn(acc[0], acc[1], o, lse)
            else:
                results[item] = (o, lse)                        # a helper's partial: travels back one stage later
        for r in reqs:
            r.wait()
        for _, op, tensor, peer, item in (tuple(int(v) for v in c) for c in mine):
            if op != SAP_OP_COPY:
                continue
            buf = recv.pop((tensor, peer, item))
            if tensor == SAP_T_Q:
                q_buf[item] = buf
            elif tensor == SAP_T_KV:
                kv_buf[item] = buf
            else:                                               # copy and rescale
                o, lse = unpack_o(buf)
                acc = (o, lse) if acc is None else merge_fn(acc[0], acc[1], o, lse)
    assert not q_buf and not kv_buf and not results, "every transferred tensor was consumed"
    return acc if acc is not None else (None, None)



def sap_execute_bwd(q_shard, do_pack, kv_shard, plan: Plan, slots: np.ndarray, rank: int, bwd_fn: Callable, group=None):
    """Replays rank `rank`'s backward code list (sap_plan_codegen_bwd).  q_shard [n,Hq,d]; do_pack: this rank's dO
    rows with their LSE and D packed in one tensor (it travels as the `do` tensor of Table 1); kv_shard [2,n,Hkv,d].
    bwd_fn(item, q_shard, do_pack, kv_shard) -> (dq [n,Hq,d], dkv [2,n,Hkv,d]) : the item's contributions to the rows
    of chunk q_chunk(item) and to the keys of chunk kv_chunk(item), as tensors torch.distributed can send.
    Returns this rank's (dq, dkv): own contributions plus everything the COPY codes added."""
    import torch
    import torch.distributed as dist

    codes = plan.codegen(slots, rank, backward=True)
    items = plan.items
    dq_acc, dkv_acc = None, None
    bufs, results = {}, {}                      # (tensor, item) -> received operand; (tensor, item) -> contribution to send
    add = lambda acc, t: t.clone() if acc is None else acc + t
    for st in sorted(set(int(c[0]) for c in codes)):
        mine = [tuple(int(v) for v in c) for c in codes if int(c[0]) == st]
        ops, recv = [], {}
        for _, op, tensor, peer, item in mine:
            if op == SAP_OP_SEND:
                payload = {SAP_T_Q: q_shard, SAP_T_DO: do_pack, SAP_T_KV: kv_shard}.get(tensor)
                if payload is None:
                    payload = results.pop((tensor, item))
                ops.append(dist.P2POp(dist.isend, payload.contiguous(), peer, group))
            elif op == SAP_OP_RECV:
                like = {SAP_T_Q: q_shard, SAP_T_DO: do_pack, SAP_T_KV: kv_shard, SAP_T_DQ: q_shard, SAP_T_DKV: kv_shard}[tensor]
                recv[(tensor, item)] = torch.empty_like(like)
                ops.append(dist.P2POp(dist.irecv, recv[(tensor, item)], peer, group))
        reqs = dist.batch_isend_irecv(ops) if ops else []
        for _, op, tensor, peer, item in mine:
            if op != SAP_OP_COMPUTING:
                continue
            i, j = int(items[item, 0]), int(items[item, 1])
            qs = q_shard if i == rank else bufs.pop((SAP_T_Q, item))
            dos = do_pack if i == rank else bufs.pop((SAP_T_DO, item))
            kv = kv_shard if j == rank else bufs.pop((SAP_T_KV, item))
            dq, dkv = bwd_fn(item, qs, dos, kv)
            if i == rank:
                dq_acc = add(dq_acc, dq)
            else:
                results[(SAP_T_DQ, item)] = dq      # travels back to the rank of the rows one stage later
            if j == rank:
                dkv_acc = add(dkv_acc, dkv)
            else:
                results[(SAP_T_DKV, item)] = dkv    # travels back to the rank of the keys one stage later
        for r in reqs:
            r.wait()
        for _, op, tensor, peer, item in mine:
            if op != SAP_OP_COPY:
                continue
            buf = recv.pop((tensor, item))
            if tensor == SAP_T_DQ:
                dq_acc = add(dq_acc, buf)
            elif tensor == SAP_T_DKV:
                dkv_acc = add(dkv_acc, buf)
            else:
                bufs[(tensor, item)] = buf
    assert not bufs and not results, "every transferred tensor was consumed"
    return dq_acc, dkv_acc
