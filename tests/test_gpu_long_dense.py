"""Dense-dO dK/dV on the EARLY and MIDDLE key columns of a long document (parity finding 2): a column s of a
document needs every later row t >= s, so column 0 of a 128K-token document (the length of BASELINE.json configs[3])
accumulates 131072 dense rows x the q-heads
of the group through every streamed tile and pipeline iteration of the backward kernel.  test_gpu_configs.py reaches
those columns only with a sparse dO (the oracle needs all row statistics: O(L^2) on the CPU, about two minutes on the
GPU box's host cores), which is why this case is one document, one KV group of two q-heads.

Tolerance: BASELINE.json north_star per element plus the norm-relative head-vector rule (tests/parity.py), which is
the one that bites here: |dK|, |dV| elements of an early column are O(1) but out / dQ rows are ~1e-2."""
import numpy as np
import pytest
import torch

import paper_2606_30460_b200 as sap
from oracle import oracle
from paper_2606_30460_b200.workloads import custom_workload, make_qkv
from parity import check_close, check_lse, to_np, row_scale, col_scale

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


def test_dense_dout_early_and_middle_columns_of_a_128k_document():
    L = 131072
    w = custom_workload([L], 16, 2, 1, 128, name="long_dense_128k")
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    dq, dk, dv = sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale)
    torch.cuda.synchronize()
    for name, t in (("out", out), ("lse", lse), ("dq", dq), ("dk", dk), ("dv", dv)):
        assert bool(torch.isfinite(t).all()), f"{name}: non-finite values"
    args = (to_np(q), to_np(k), to_np(v))
    # early, middle (both sides of a chunk boundary and of a 256-key pair-tile boundary) and last columns
    cols = np.concatenate([np.arange(0, 128), np.arange(L // 2 - 64, L // 2 + 64), np.arange(L // 4 + 128 - 32, L // 4 + 128 + 32),
                           np.arange(L - 64, L)])
    dk_ref, dv_ref = oracle.attn_bwd_dkv(*args, to_np(do), w.cu_seqlens, w.softmax_scale, cols=cols)
    cols_t = torch.from_numpy(cols).cuda()
    nr = col_scale(w.cu_seqlens, cols)
    check_close(to_np(dk[cols_t]), dk_ref, f"dk[{len(cols)} early / middle / last columns]", nr)
    check_close(to_np(dv[cols_t]), dv_ref, f"dv[{len(cols)} early / middle / last columns]", nr)
    # rows: first rows, chunk and tile boundaries, the last rows (131072 visible keys)
    rng = np.random.default_rng(7)
    rows = np.unique(np.concatenate([np.arange(0, 4), np.arange(L // 2 - 2, L // 2 + 2), np.arange(L - 8, L),
                                     rng.integers(0, L, size=96)]))
    rows_t = torch.from_numpy(rows).cuda()
    nk = row_scale(w.cu_seqlens, rows)
    o_ref, l_ref = oracle.attn_fwd(*args, w.cu_seqlens, w.softmax_scale, rows=rows)
    check_close(to_np(out[rows_t]), o_ref, "out", nk)
    check_lse(to_np(lse[:, rows_t]).T, l_ref, "lse")
    dq_ref = oracle.attn_bwd_dq(*args, to_np(do), w.cu_seqlens, w.softmax_scale, rows=rows)
    check_close(to_np(dq[rows_t]), dq_ref, "dq", nk)
