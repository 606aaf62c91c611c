"""SURVEY 8(f) NEXT-1 (host side): the forward pass with REAL ranks, one sequence chunk per rank.

The paper's execute side (Table 1 :85-98): rank i owns Q_i, K_i, V_i (n = N/P rows, :59); K/V shards
travel rank to rank, every kept chunk pair (i, j) is one `computing` instruction on rank i, and the partial
results are merged "in an online manner" (:59).  Which shards travel is decided by the plan, not by the ring: a
rank sends its K/V shard only to the ranks whose plan has a non-SKIP item against it (the "trim redundant
communication" of :106), and each ring step is ONE batched isend/irecv that covers the whole group, which is what
lets NCCL coalesce it (:124).  Step s+1's transfers are posted before step s is computed (:120-122).

On B200 nodes every peer is one NVSwitch hop away, so the paper's NVLink / InfiniBand placement (:144) has no
counterpart here: the schedule is the plan's ring order and nothing else.

This module is the exchange schedule plus argument marshalling.  The arithmetic is behind two callables:
`partial_fn(item_index, k_shard, v_shard) -> (o [n,Hq,d] fp32, lse [Hq,n] fp32)` for this rank's rows and
`merge_fn(o_a, lse_a, o_b, lse_b) -> (o, lse)`.  `cuda_fns()` builds them from the C-ABI kernels
(`sap_attn_fwd_partial`, `sap_lse_merge`); the CPU tests (gloo, world_size 2 and 4) inject the oracle's.  It has
not run on more than one GPU (this build has one): correct by construction, covered on CPU.
"""
from __future__ import annotations

from typing import Callable, List, Optional, Tuple

from .api import Plan, SAP_MASK_SKIP


def step_peers(plan: Plan, rank: int, step: int) -> Tuple[Optional[int], Optional[int]]:
    """(dst, src) of ring step `step` >= 1 for `rank`: dst = rank + step gets my K/V shard iff its plan has a
    non-SKIP item against chunk `rank`; src = rank - step sends me its shard iff my plan has one against it."""
    P = plan.n_chunks
    km = plan.kind_map
    dst = rank + step if rank + step < P and km[rank + step, rank] != SAP_MASK_SKIP else None
    src = rank - step if rank - step >= 0 and km[rank, rank - step] != SAP_MASK_SKIP else None
    return dst, src


def schedule(plan: Plan) -> List[List[Tuple[int, int]]]:
    """All (src, dst) transfers per ring step, for the whole group (the same list on every rank)."""
    P = plan.n_chunks
    out = []
    for step in range(1, P):
        out.append([(r, r + step) for r in range(P - step) if plan.kind_map[r + step, r] != SAP_MASK_SKIP])
    return out


def sap_ring_fwd(kv_shard, plan: Plan, rank: int, partial_fn: Callable, merge_fn: Callable, group=None):
    """Forward of chunk `rank`.  kv_shard: this rank's stacked K/V shard [2, n, Hkv, d] (any device / dtype
    torch.distributed can send).  Returns the merged (o, lse) of this rank's rows."""
    import torch
    import torch.distributed as dist

    P = plan.n_chunks
    assert dist.get_world_size(group) == P, "one rank per sequence chunk"
    # `rank` and the plan's chunk indices are ranks INSIDE `group` (HSAP runs the SAP ring over an inter-group
    # sub-communicator); P2POp wants global ranks
    glob = (lambda r: r) if group is None else (lambda r: dist.get_global_rank(group, r))
    items = plan.items
    co = plan.chunk_offsets
    my_items = {int(items[x, 1]): x for x in range(int(co[rank]), int(co[rank + 1]))}   # kv_chunk -> item index

    def post(step):
        """One batched isend/irecv for ring step `step`; returns (requests, receive buffer or None)."""
        dst, src = step_peers(plan, rank, step)
        ops, buf = [], None
        if dst is not None:
            ops.append(dist.P2POp(dist.isend, kv_shard, glob(dst), group))
        if src is not None:
            buf = torch.empty_like(kv_shard)
            ops.append(dist.P2POp(dist.irecv, buf, glob(src), group))
        return (dist.batch_isend_irecv(ops) if ops else []), buf

    nxt = post(1) if P > 1 else ([], None)
    o, lse = partial_fn(my_items[rank], kv_shard[0], kv_shard[1])            # step 0: the diagonal block
    for step in range(1, P):
        reqs, buf = nxt
        nxt = post(step + 1) if step + 1 < P else ([], None)                 # next step's transfer overlaps this compute
        for r in reqs:
            r.wait()
        j = rank - step
        if buf is not None and j in my_items:
            po, pl = partial_fn(my_items[j], buf[0], buf[1])
            o, lse = merge_fn(o, lse, po, pl)
    return o, lse


def cuda_fns(q_shard, cu_seqlens_dev, plan: Plan, rank: int, softmax_scale: Optional[float] = None):
    """(partial_fn, merge_fn) on the C-ABI kernels.  The kernels address tokens globally; the shards are handed over as
    executor.ShardView (base pointer moved back by the shard's first row) and the forward `computing` entry
    sap_attn_fwd_items touches only the Q tiles of the item, so a rank holds its own Q rows, the K/V shard in flight
    and one partial result: O(N/P) memory and work per item (only the per-row LSE buffer, 4 bytes per row and head,
    is full length: the library's [Hq, N] layout).

    That holds when the shard length n = N/P is a multiple of the 128-row tile (sap.h, shard-pointer contract).  The
    kernels move whole 128-row boxes that start on multiples of 128, so with any other n a box of the first or last
    tile of a shard reaches rows of the neighbouring shard - memory a shard-sized buffer does not have.  Then the
    callables fall back to zero-filled full-length buffers with the shard copied into its rows (O(N) memory, same
    result: rows outside the shard are masked by the item's row and key ranges)."""
    import torch
    from . import api
    from .executor import ShardView, shard_view_ok

    n, Hq, d = q_shard.shape
    N = plan.n_tokens
    dev = q_shard.device
    lo, hi = rank * n, (rank + 1) * n
    lse_full = torch.empty((Hq, N), dtype=torch.float32, device=dev)
    by_view = shard_view_ok(n)

    def place(shard, row0):
        """the tensor the kernels see: a view of the shard, or a full-length copy when views are not safe"""
        if by_view:
            return ShardView(shard.contiguous(), row0, N)
        full = torch.zeros((N,) + tuple(shard.shape[1:]), dtype=shard.dtype, device=dev)
        full[row0:row0 + shard.shape[0]] = shard
        return full

    qg = place(q_shard, lo)

    def partial_fn(item, k_shard, v_shard):
        j = int(plan.items[item, 1])
        Hkv = k_shard.shape[1]
        o = torch.zeros((n, Hq, d), dtype=torch.float32, device=dev)   # Q tiles the item does not touch: the (0, -inf) identity
        lse_full[:, lo:hi] = float("-inf")
        og = place(o, lo)
        api.sap_attn_fwd_items(qg, place(k_shard, j * n), place(v_shard, j * n), cu_seqlens_dev, plan, item, item + 1, og,
                               lse_full, Hq, Hkv, d, softmax_scale=softmax_scale)
        if not by_view:
            o = og[lo:hi].contiguous()
        return o, lse_full[:, lo:hi].contiguous()

    def merge_fn(o_a, lse_a, o_b, lse_b):
        return api.sap_lse_merge(o_a, lse_a, o_b, lse_b)

    return partial_fn, merge_fn
