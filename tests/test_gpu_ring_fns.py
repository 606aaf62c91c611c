"""The CUDA callables of paper_2606_30460_b200.ring (per-item partial on a received K/V shard + LSE merge), driven
rank by rank in ONE process on one GPU (no process group: the exchange itself is covered on CPU by
tests/test_ring_gloo.py).  Result per rank == the fused forward == the oracle."""
import numpy as np
import pytest
import torch

import paper_2606_30460_b200 as sap
from oracle import oracle
from paper_2606_30460_b200 import ring
from paper_2606_30460_b200.workloads import custom_workload, make_qkv
from parity import check_close, check_lse, to_np

pytestmark = pytest.mark.gpu


# P = 5 over 2050 tokens: shards of 410 rows, not a multiple of the 128-row tile - the callables must then hand the kernels
# full-length buffers (sap.h, shard-pointer contract), since a tile's box would leave a shard-sized allocation
@pytest.mark.parametrize("P,lens", [(1, [700, 1100, 248]), (4, [700, 1100, 248]), (5, [700, 1100, 250])])
def test_rank_by_rank_partials_equal_fused(P, lens):
    w = custom_workload(lens, P, 4, 2, 128)
    q, k, v = make_qkv(w, device="cuda", with_dout=False)
    plan = sap.sap_plan(w.cu_seqlens, P)
    cu = plan.cu_seqlens_dev("cuda")
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    o_ref, l_ref = oracle.attn_fwd(to_np(q), to_np(k), to_np(v), w.cu_seqlens, w.softmax_scale)
    n = w.n_tokens // P
    for r in range(P):
        lo, hi = r * n, (r + 1) * n
        partial_fn, merge_fn = ring.cuda_fns(q[lo:hi], cu, plan, r, softmax_scale=w.softmax_scale)
        o = l = None
        for x in range(int(plan.chunk_offsets[r]), int(plan.chunk_offsets[r + 1])):   # ring order
            j = int(plan.items[x, 1])
            po, pl = partial_fn(x, k[j * n:(j + 1) * n], v[j * n:(j + 1) * n])
            o, l = (po, pl) if o is None else merge_fn(o, l, po, pl)
        torch.cuda.synchronize()
        check_close(to_np(o), o_ref[lo:hi], f"P={P} rank {r} out")
        check_lse(to_np(l).T, l_ref[lo:hi], f"P={P} rank {r} lse")
        check_close(to_np(o), to_np(out[lo:hi]), f"P={P} rank {r} vs fused")
