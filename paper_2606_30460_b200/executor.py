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
    # `rank` and the peers in the code list are ranks inside `group`; P2POp wants global ranks
    glob = (lambda r: r) if group is None else (lambda r: dist.get_global_rank(group, r))
    stages = sorted(set(int(c[0]) for c in codes))
    q_buf, kv_buf, results, acc = {}, {}, {}, None           # per item: received q / kv; computed partials to send
    for st in stages:
        mine = [c for c in codes if int(c[0]) == st]
        ops, recv = [], {}
        for _, op, tensor, peer, item in (tuple(int(v) for v in c) for c in mine):
            if op == SAP_OP_SEND:
                payload = q_shard if tensor == SAP_T_Q else kv_shard if tensor == SAP_T_KV else pack_o(*results.pop(item))
                ops.append(dist.P2POp(dist.isend, payload.contiguous(), glob(peer), group))
            elif op == SAP_OP_RECV:
                like = q_shard if tensor == SAP_T_Q else kv_shard if tensor == SAP_T_KV else o_template
                recv[(tensor, peer, item)] = torch.empty_like(like)
                ops.append(dist.P2POp(dist.irecv, recv[(tensor, peer, item)], glob(peer), group))
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



def sap_execute_bwd(q_shard, do_pack, kv_shard, plan: Plan, slots: np.ndarray, rank: int, bwd_fn: Callable, group=None,
                    add_fn: Callable = None):
    """Replays rank `rank`'s backward code list (sap_plan_codegen_bwd).  q_shard [n,Hq,d]; do_pack: this rank's dO
    rows with their LSE and D packed in one tensor (it travels as the `do` tensor of Table 1); kv_shard [2,n,Hkv,d].
    bwd_fn(item, q_shard, do_pack, kv_shard) -> (dq [n,Hq,d], dkv [2,n,Hkv,d]) : the item's contributions to the rows
    of chunk q_chunk(item) and to the keys of chunk kv_chunk(item), as tensors torch.distributed can send.
    add_fn(acc, t) adds a contribution into a gradient in place (COPY of a received dq / dkv, Table 1); the default is
    the tensor library's add for the CPU schedule tests, on a GPU pass api.sap_axpy (LocalExecutor does).
    Returns this rank's (dq, dkv): own contributions plus everything the COPY codes added."""
    import torch
    import torch.distributed as dist

    codes = plan.codegen(slots, rank, backward=True)
    items = plan.items
    glob = (lambda r: r) if group is None else (lambda r: dist.get_global_rank(group, r))
    dq_acc, dkv_acc = None, None
    bufs, results = {}, {}                      # (tensor, item) -> received operand; (tensor, item) -> contribution to send
    add_fn = add_fn or (lambda acc, t: acc.add_(t))
    add = lambda acc, t: t.clone() if acc is None else add_fn(acc, t)
    for st in sorted(set(int(c[0]) for c in codes)):
        mine = [tuple(int(v) for v in c) for c in codes if int(c[0]) == st]
        ops, recv = [], {}
        for _, op, tensor, peer, item in mine:
            if op == SAP_OP_SEND:
                payload = {SAP_T_Q: q_shard, SAP_T_DO: do_pack, SAP_T_KV: kv_shard}.get(tensor)
                if payload is None:
                    payload = results.pop((tensor, item))
                ops.append(dist.P2POp(dist.isend, payload.contiguous(), glob(peer), group))
            elif op == SAP_OP_RECV:
                like = {SAP_T_Q: q_shard, SAP_T_DO: do_pack, SAP_T_KV: kv_shard, SAP_T_DQ: q_shard, SAP_T_DKV: kv_shard}[tensor]
                recv[(tensor, item)] = torch.empty_like(like)
                ops.append(dist.P2POp(dist.irecv, recv[(tensor, item)], glob(peer), group))
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


# ======================================================================================================================
# One-GPU replay: the P ranks are emulated in one process (BASELINE.json north_star: "the P ranks are emulated as P
# sequence chunks in HBM"), every rank's code list is executed stage by stage, the transport is a device copy into the
# receiver's staging buffer, and every arithmetic step is a kernel behind the C ABI.
# ======================================================================================================================
class ShardView:
    """A shard [n, H, d] that the kernels address with GLOBAL token indices: data_ptr() is moved back by `row0` rows,
    so that row t of the whole tensor lands on row t - row0 of the shard.  The kernels touch only the rows their tile
    program names (the shard's), so a rank needs memory for one shard, not for the sequence."""

    def __init__(self, shard, row0: int, n_tokens: int):
        assert shard.is_contiguous()
        self._t, self._row0 = shard, int(row0)
        self.shape = (int(n_tokens),) + tuple(shard.shape[1:])
        self.dtype, self.device, self.is_cuda = shard.dtype, shard.device, shard.is_cuda

    def is_contiguous(self):
        return True

    def data_ptr(self):
        return self._t.data_ptr() - self._row0 * self._t.stride(0) * self._t.element_size()


def shard_view_ok(n: int, head_dim: int = 0, backward: bool = False) -> bool:
    """May shards of n rows be handed to the kernels as ShardViews?  (sap.h, shard-pointer contract.)  The kernels move
    whole tiles that start on multiples of the tile length - 128 rows; 256 keys for the head_dim-128 backward, which
    runs on CTA pairs - so a shard boundary inside a tile makes a box reach into the neighbouring shard, outside a
    shard-sized allocation."""
    tile = 256 if (backward and head_dim == 128) else 128
    return n > 0 and n % tile == 0


def _ws_bytes(plan, Hq, Hkv, d):
    from . import api
    return api.sap_workspace_bytes(plan, Hq, Hkv, d, api.SAP_PASS_BWD)


def _max_inflight(code_lists, tensor_kinds):
    """largest number of same-kind RECVs one rank has in one stage: the 'fixed multiple' of a shard the staging area
    needs"""
    worst = 1
    for codes in code_lists:
        count = {}
        for st, op, tensor, peer, item in codes.tolist():
            if op == SAP_OP_RECV and tensor in tensor_kinds:
                count[(st, tensor)] = count.get((st, tensor), 0) + 1
        worst = max([worst] + list(count.values()))
    return worst


class LocalExecutor:
    """Replays the jitted code lists of all P ranks on ONE GPU (forward and backward).

    Per rank: its own shards (views of the caller's tensors), one compute buffer per operand kind (q, kv, do) that COPY
    fills from the staging area ("copy from the communication buffer to the compute buffer"), a staging
    area of a fixed number of shard-sized slots per tensor kind allocated ONCE (:140-142), and the running result.
    SEND / RECV of a stage are matched across ranks and executed as device copies before the stage's COMPUTING codes,
    COPY codes after them, exactly in the order of the lists (sap_plan_codegen / sap_plan_codegen_bwd).  COMPUTING
    asserts that its operands are present: an illegal schedule fails here, not in the numerics."""

    def __init__(self, plan: Plan, slots: np.ndarray, n_q_heads: int, n_kv_heads: int, head_dim: int, device,
                 softmax_scale=None):
        import torch
        self.plan, self.slots = plan, np.ascontiguousarray(slots, dtype=np.int32)
        self.P, self.N = plan.n_chunks, plan.n_tokens
        self.n = self.N // self.P
        self.Hq, self.Hkv, self.d, self.dev = n_q_heads, n_kv_heads, head_dim, device
        self.scale = float(head_dim) ** -0.5 if softmax_scale is None else float(softmax_scale)
        self.items = plan.items
        # K/V tiles of the per-item backward are 256 keys (head_dim 128) or 128 keys wide from token 0: a rank's shard-sized
        # dK / dV buffer holds whole tiles only if the chunk length is a multiple of that
        assert shard_view_ok(self.n, head_dim, backward=True), "chunk length must be a multiple of the K/V tile"
        self.fwd_codes = [plan.codegen(self.slots, r) for r in range(self.P)]
        self.bwd_codes = [plan.codegen(self.slots, r, backward=True) for r in range(self.P)]
        n, Hq, Hkv, d, P = self.n, n_q_heads, n_kv_heads, head_dim, self.P
        bf, f32 = torch.bfloat16, torch.float32
        e = lambda *shape, dtype=bf: torch.empty(shape, dtype=dtype, device=device)
        kq = _max_inflight(self.fwd_codes + self.bwd_codes, (SAP_T_Q,))
        kkv = _max_inflight(self.fwd_codes + self.bwd_codes, (SAP_T_KV,))
        ko = _max_inflight(self.fwd_codes, (SAP_T_O,))
        kdo = _max_inflight(self.bwd_codes, (SAP_T_DO,))
        kdq = _max_inflight(self.bwd_codes, (SAP_T_DQ,))
        kdkv = _max_inflight(self.bwd_codes, (SAP_T_DKV,))
        self.staging_slots = {"q": kq, "kv": kkv, "o": ko, "do": kdo, "dq": kdq, "dkv": kdkv}
        # fixed buffers, allocated once for all P emulated ranks (one of each per rank)
        self.stage_q = e(P, kq, n, Hq, d); self.stage_kv = e(P, kkv, 2, n, Hkv, d)
        self.stage_o = e(P, ko, n, Hq, d, dtype=f32); self.stage_ol = e(P, ko, Hq, n, dtype=f32)
        self.stage_do = e(P, kdo, n, Hq, d); self.stage_dol = e(P, kdo, 2, Hq, n, dtype=f32)      # dO with LSE and D
        self.stage_dq = e(P, kdq, n, Hq, d, dtype=f32); self.stage_dkv = e(P, kdkv, 2, n, Hkv, d)
        self.comp_q = e(P, n, Hq, d); self.comp_kv = e(P, 2, n, Hkv, d)
        self.comp_do = e(P, n, Hq, d); self.comp_dol = e(P, 2, Hq, n, dtype=f32)
        self.part_o = e(n, Hq, d, dtype=f32); self.part_l = e(Hq, self.N, dtype=f32)              # one partial result
        self.part_lc = e(Hq, n, dtype=f32)                                                         # its LSE rows, shard-sized
        self.scratch_dkv = e(2, n, Hkv, d)
        # what a rank computed for another rank waits here until the next stage's SEND: a rank runs one item per stage and
        # its result leaves one stage later, so one slot per rank and kind is enough
        self.out_o = e(P, n, Hq, d, dtype=f32); self.out_ol = e(P, Hq, n, dtype=f32)
        self.out_dq = e(P, n, Hq, d, dtype=f32); self.out_dkv = e(P, 2, n, Hkv, d)
        # running results of all P ranks, and the backward workspaces.  The C ABI lays a workspace out as D [Hq, N] followed by
        # the accumulator [N, Hq, d] from ONE base pointer and addresses both by global token, so even the helper's scratch
        # workspace has to be full length (a rank proper would need its own rows plus one shard); they are allocated once.
        self.acc_o = e(P, n, Hq, d, dtype=f32); self.acc_l = e(P, Hq, n, dtype=f32)
        need = _ws_bytes(plan, Hq, Hkv, d)
        self.ws_own = torch.empty(need, dtype=torch.uint8, device=device)     # owners' D and dQ accumulator rows
        self.ws_help = torch.empty(need, dtype=torch.uint8, device=device)    # scratch of the rank that helps another
        self.dkv_tot = e(2, self.N, Hkv, d, dtype=f32)
        self.mem_marks = []       # torch.cuda.memory_allocated() at the start of every stage of the last replay (tests)

    # ------------------------------------------------------------------------------------------------ helpers
    def _walk(self, code_lists, on_transfer, on_compute, on_copy):
        import torch
        stages = sorted(set(int(c[0]) for codes in code_lists for c in codes))
        self.mem_marks = []
        for st in stages:
            self.mem_marks.append(torch.cuda.memory_allocated(self.dev))
            per_rank = [[tuple(int(v) for v in c) for c in codes if int(c[0]) == st] for codes in code_lists]
            sends = {(tensor, r, peer, item) for r, mine in enumerate(per_rank) for _, op, tensor, peer, item in mine if op == SAP_OP_SEND}
            recvs = [(tensor, peer, r, item) for r, mine in enumerate(per_rank) for _, op, tensor, peer, item in mine if op == SAP_OP_RECV]
            assert sends == set(recvs) and len(recvs) == len(set(recvs)), f"stage {st}: SEND / RECV codes do not pair up"
            slot_of = {}
            for tensor, src, dst, item in recvs:                    # the batched isend/irecv of the stage
                k = sum(1 for (t2, _, d2, _) in slot_of if t2 == tensor and d2 == dst)
                slot_of[(tensor, src, dst, item)] = k
                on_transfer(tensor, src, dst, item, k)
            for r, mine in enumerate(per_rank):
                for _, op, tensor, peer, item in mine:
                    if op == SAP_OP_COMPUTING:
                        on_compute(r, item)
            for r, mine in enumerate(per_rank):
                for _, op, tensor, peer, item in mine:
                    if op == SAP_OP_COPY:
                        on_copy(r, tensor, peer, item, slot_of[(tensor, peer, r, item)])
        self.mem_marks.append(torch.cuda.memory_allocated(self.dev))

    # ------------------------------------------------------------------------------------------------ forward
    def forward(self, q, k, v, cu_seqlens_dev):
        """q [N,Hq,d], k, v [N,Hkv,d] bf16 on the device (rank r owns rows [r n, (r+1) n)).  Returns out bf16 [N,Hq,d],
        lse fp32 [Hq,N]."""
        import torch
        from . import api
        n, N, P, Hq = self.n, self.N, self.P, self.Hq
        own_q = lambda r: q[r * n:(r + 1) * n]
        own_kv = lambda r: (k[r * n:(r + 1) * n], v[r * n:(r + 1) * n])
        acc_o, acc_l = self.acc_o.zero_(), self.acc_l.fill_(float("-inf"))
        have_q, have_kv, results = {}, {}, {}      # (rank, item) -> operand in the compute buffer; helper partials

        def merge(r, item, o, l):
            # only the 128-row Q tiles the item touches hold a partial result (sap_attn_fwd_items leaves the others alone)
            rb = (int(self.items[item, 6]) - r * n) // 128 * 128
            re = min(n, -(-(int(self.items[item, 7]) - r * n) // 128) * 128)
            api.sap_lse_merge(acc_o[r], acc_l[r], o, l, row_begin=rb, row_end=re, o_out=acc_o[r], lse_out=acc_l[r])

        def on_transfer(tensor, src, dst, item, slot):
            if tensor == SAP_T_Q:
                self.stage_q[dst, slot].copy_(own_q(src))
            elif tensor == SAP_T_KV:
                kk, vv = own_kv(src)
                self.stage_kv[dst, slot, 0].copy_(kk); self.stage_kv[dst, slot, 1].copy_(vv)
            else:
                o, l = results.pop((src, item))
                self.stage_o[dst, slot].copy_(o); self.stage_ol[dst, slot].copy_(l)

        def on_compute(r, item):
            i, j = int(self.items[item, 0]), int(self.items[item, 1])
            assert r in (i, j)
            if i == r:
                qs = own_q(r)
            else:
                assert have_q.pop((r, item), False), f"rank {r}: Q of item {item} is not in the compute buffer"
                qs = self.comp_q[r]
            if j == r:
                ks, vs = own_kv(r)
            else:
                assert have_kv.pop((r, item), False), f"rank {r}: K/V of item {item} is not in the compute buffer"
                ks, vs = self.comp_kv[r, 0], self.comp_kv[r, 1]
            qg, kg, vg = ShardView(qs.contiguous(), i * n, N), ShardView(ks.contiguous(), j * n, N), ShardView(vs.contiguous(), j * n, N)
            api.sap_attn_fwd_items(qg, kg, vg, cu_seqlens_dev, self.plan, item, item + 1, ShardView(self.part_o, i * n, N),
                                          self.part_l, Hq, self.Hkv, self.d, softmax_scale=self.scale)
            o, l = self.part_o, self.part_lc.copy_(self.part_l[:, i * n:(i + 1) * n])
            if i == r:
                merge(r, item, o, l)
            else:                                            # a helper's partial: travels back one stage later
                assert not any(key[0] == r for key in results), f"rank {r}: its previous partial result has not been sent yet"
                results[(r, item)] = (self.out_o[r].copy_(o), self.out_ol[r].copy_(l))

        def on_copy(r, tensor, peer, item, slot):
            if tensor == SAP_T_Q:
                self.comp_q[r].copy_(self.stage_q[r, slot]); have_q[(r, item)] = True
            elif tensor == SAP_T_KV:
                self.comp_kv[r].copy_(self.stage_kv[r, slot]); have_kv[(r, item)] = True
            else:                                            # copy and rescale
                merge(r, item, self.stage_o[r, slot], self.stage_ol[r, slot])

        self._walk(self.fwd_codes, on_transfer, on_compute, on_copy)
        assert not have_q and not have_kv and not results, "every transferred tensor was consumed"
        out = torch.empty_like(q)
        api.sap_axpy(out, acc_o.reshape(N, Hq, self.d), 1.0, accumulate=False)
        return out, acc_l.permute(1, 0, 2).reshape(Hq, N).contiguous()

    # ------------------------------------------------------------------------------------------------ backward
    def backward(self, dout, q, k, v, out, lse, cu_seqlens_dev):
        """Returns dq [N,Hq,d], dk, dv [N,Hkv,d] bf16."""
        import torch
        from . import api
        n, N, P, Hq, Hkv, d = self.n, self.N, self.P, self.Hq, self.Hkv, self.d
        ws_own, ws_help = self.ws_own, self.ws_help
        acc_off = ((N * Hq * 4 + 255) // 256) * 256
        dsum = lambda ws: ws[:N * Hq * 4].view(torch.float32).view(Hq, N)
        dqacc = lambda ws: ws[acc_off:acc_off + N * Hq * d * 4].view(torch.float32).view(N, Hq, d)
        for r in range(P):   # every rank: D of its rows, zero its accumulator rows (sap_attn_bwd_begin)
            api.sap_attn_bwd_begin(dout, out, self.plan, r, r + 1, Hkv, ws_own)
        dkv_tot = self.dkv_tot.zero_()
        have, results = {}, {}
        own = lambda t, r: t[r * n:(r + 1) * n]

        def on_transfer(tensor, src, dst, item, slot):
            if tensor == SAP_T_Q:
                self.stage_q[dst, slot].copy_(own(q, src))
            elif tensor == SAP_T_KV:
                self.stage_kv[dst, slot, 0].copy_(own(k, src)); self.stage_kv[dst, slot, 1].copy_(own(v, src))
            elif tensor == SAP_T_DO:                          # dO rows with their LSE and D
                self.stage_do[dst, slot].copy_(own(dout, src))
                self.stage_dol[dst, slot, 0].copy_(lse[:, src * n:(src + 1) * n]); self.stage_dol[dst, slot, 1].copy_(dsum(ws_own)[:, src * n:(src + 1) * n])
            elif tensor == SAP_T_DQ:
                self.stage_dq[dst, slot].copy_(results.pop((src, SAP_T_DQ, item)))
            else:
                self.stage_dkv[dst, slot].copy_(results.pop((src, SAP_T_DKV, item)))

        def on_compute(r, item):
            i, j = int(self.items[item, 0]), int(self.items[item, 1])
            assert r in (i, j)
            if i == r:
                qs, dos, ws, lse_g = own(q, r), own(dout, r), ws_own, lse
            else:       # helper: Q, dO (with LSE, D) of chunk i arrived; contributions to dQ go to scratch rows of chunk i
                assert have.pop((r, SAP_T_Q, item), False) and have.pop((r, SAP_T_DO, item), False), f"rank {r}: q / do of item {item} missing"
                qs, dos, ws = self.comp_q[r], self.comp_do[r], ws_help
                lse_g = self.part_l
                lse_g[:, i * n:(i + 1) * n].copy_(self.comp_dol[r, 0]); dsum(ws)[:, i * n:(i + 1) * n].copy_(self.comp_dol[r, 1])
                dqacc(ws)[i * n:(i + 1) * n].zero_()
            if j == r:
                ks, vs = own(k, r), own(v, r)
            else:
                assert have.pop((r, SAP_T_KV, item), False), f"rank {r}: K/V of item {item} missing"
                ks, vs = self.comp_kv[r, 0], self.comp_kv[r, 1]
            view = lambda t, c: ShardView(t.contiguous(), c * n, N)
            api.sap_attn_bwd_items(view(dos, i), view(qs, i), view(ks, j), view(vs, j), lse_g, cu_seqlens_dev, self.plan, item, item + 1,
                                   view(self.scratch_dkv[0], j), view(self.scratch_dkv[1], j), ws, softmax_scale=self.scale)
            it = self.items[item]
            kb, ke = int(it[8]) - j * n, int(it[9]) - j * n      # the item's key rows inside chunk j (other rows of touched tiles: zero)
            if j == r:
                api.sap_axpy(dkv_tot[0, j * n + kb:j * n + ke], self.scratch_dkv[0, kb:ke], 1.0)
                api.sap_axpy(dkv_tot[1, j * n + kb:j * n + ke], self.scratch_dkv[1, kb:ke], 1.0)
            else:
                assert not any(key[0] == r for key in results), f"rank {r}: its previous contribution has not been sent yet"
                c = self.out_dkv[r].zero_(); c[:, kb:ke].copy_(self.scratch_dkv[:, kb:ke])
                results[(r, SAP_T_DKV, item)] = c
            if i != r:
                assert not any(key[0] == r for key in results), f"rank {r}: its previous contribution has not been sent yet"
                results[(r, SAP_T_DQ, item)] = self.out_dq[r].copy_(dqacc(ws)[i * n:(i + 1) * n])

        def on_copy(r, tensor, peer, item, slot):
            if tensor == SAP_T_Q:
                self.comp_q[r].copy_(self.stage_q[r, slot]); have[(r, tensor, item)] = True
            elif tensor == SAP_T_KV:
                self.comp_kv[r].copy_(self.stage_kv[r, slot]); have[(r, tensor, item)] = True
            elif tensor == SAP_T_DO:
                self.comp_do[r].copy_(self.stage_do[r, slot]); self.comp_dol[r].copy_(self.stage_dol[r, slot]); have[(r, tensor, item)] = True
            elif tensor == SAP_T_DQ:                          # a received dq contribution is added into the owner's accumulator
                api.sap_axpy(dqacc(ws_own)[r * n:(r + 1) * n], self.stage_dq[r, slot], 1.0)
            else:
                api.sap_axpy(dkv_tot[0, r * n:(r + 1) * n], self.stage_dkv[r, slot, 0], 1.0)
                api.sap_axpy(dkv_tot[1, r * n:(r + 1) * n], self.stage_dkv[r, slot, 1], 1.0)

        self._walk(self.bwd_codes, on_transfer, on_compute, on_copy)
        assert not have and not results, "every transferred tensor was consumed"
        dq = torch.empty_like(q)
        for r in range(P):
            api.sap_attn_bwd_end(self.plan, r, r + 1, dq, Hkv, ws_own, softmax_scale=self.scale)
        dk, dv = torch.empty_like(k), torch.empty_like(v)
        api.sap_axpy(dk, dkv_tot[0], 1.0, accumulate=False); api.sap_axpy(dv, dkv_tot[1], 1.0, accumulate=False)
        return dq, dk, dv
