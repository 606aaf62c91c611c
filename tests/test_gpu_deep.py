"""Deep parity run (SURVEY 8c coverage tier iv): one whole KV group of a 16K-token document, every row and every key
column against the fp64 oracle (about half a minute of oracle time on 16 host cores).  test_gpu_configs.py covers
the full-size configs with sampled rows / columns and the sparse-dO pass."""

import numpy as np
import pytest
import torch

import paper_2606_30460_b200 as sap
from oracle import oracle
from paper_2606_30460_b200.workloads import custom_workload, make_qkv
from parity import check_close, check_lse, to_np, row_scale, col_scale

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


def test_one_kv_group_of_a_16k_document_every_element():
    # 16K tokens in one document plus a short tail document, 8 chunks, one KV group (4 q-heads), d = 128
    w = custom_workload([16000, 384], 8, 4, 1, 128, name="deep_16k")
    q, k, v, do = make_qkv(w, device="cuda")
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    cu = plan.cu_seqlens_dev("cuda")
    out, lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
    dq, dk, dv = sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale)
    torch.cuda.synchronize()
    args = (to_np(q), to_np(k), to_np(v))
    o_ref, l_ref = oracle.attn_fwd(*args, w.cu_seqlens, w.softmax_scale)
    allt = np.arange(w.n_tokens)
    nk, nr = row_scale(w.cu_seqlens, allt), col_scale(w.cu_seqlens, allt)
    check_close(to_np(out), o_ref, "deep out", nk)
    check_lse(to_np(lse).T, l_ref, "deep lse")
    check_close(to_np(dq), oracle.attn_bwd_dq(*args, to_np(do), w.cu_seqlens, w.softmax_scale), "deep dq", nk)
    rdk, rdv = oracle.attn_bwd_dkv(*args, to_np(do), w.cu_seqlens, w.softmax_scale)
    check_close(to_np(dk), rdk, "deep dk", nr)
    check_close(to_np(dv), rdv, "deep dv", nr)
