"""One process per rank (ranks.ProcessRank) with TWO processes on the one GPU of the box: each
process creates the chunks it owns as exportable allocations, the descriptors travel over Unix sockets, every process
maps the whole range, launches only on its own chunk, and the phases are separated by group barriers (gloo) - no kernel
waits on another, the two processes' launches simply share the GPU.  Rank 0 then compares everything with its own
single launch: out, LSE, dK, dV bit for bit, dQ within tolerance.  With two GPUs the same code would place chunk 1 in the
other GPU's memory; that is not something this box can run."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, result_q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import sys
        sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
        import paper_2606_30460_b200 as sap
        from paper_2606_30460_b200.ranks import ProcessRank
        from paper_2606_30460_b200.workloads import custom_workload, make_qkv
        from parity import check_close, to_np
        # 65536 tokens, 4 chunks of 16384, 8 / 2 heads: D is 2 MiB, so the dQ accumulator can live with the chunk owners
        w = custom_workload([30000, 20000, 15536], 4, 8, 2, 128, name="process_ranks")
        Hq, Hkv, d = w.n_q_heads, w.n_kv_heads, w.head_dim
        q, k, v, do = make_qkv(w, device="cuda")                  # every process can generate the (seeded) inputs
        # two chunks of memory per rank (rank 0: chunks 0-1, rank 1: chunks 2-3); the launches are balanced by visible pairs
        # (separately for q-chunks and kv-chunks), so a rank also launches on chunks whose memory belongs to the other process
        pr = ProcessRank(w.cu_seqlens, rank, world, device=0, n_chunks=w.n_chunks)
        assert pr.owned == ([0, 1] if rank == 0 else [2, 3])
        assert set(pr.launch) != set(pr.owned) or set(pr.launch_kv) != set(pr.owned)
        sq, sdo, so, sdq = (pr.tensor((Hq, d), torch.bfloat16) for _ in range(4))
        sk, sv, sdk, sdv = (pr.tensor((Hkv, d), torch.bfloat16) for _ in range(4))
        slse = pr.shared((Hq, w.n_tokens), torch.float32)
        from paper_2606_30460_b200.ranks import workspace_units
        assert workspace_units(w.n_tokens, w.n_chunks, Hq, d, sap.Stitched.granularity(0)) == (2 << 20, 32)
        ws = pr.workspace(Hq, Hkv, d)                             # accumulator rows of chunk c in the memory of c's owner
        rows = pr.own_rows()
        for dst, src in ((sq, q), (sk, k), (sv, v), (sdo, do)):    # a rank fills only the rows it owns
            dst[rows].copy_(src[rows])
        for t in (so, sdq, sdk, sdv):
            t[rows].fill_(float("nan"))
        if rank == 0:
            slse.fill_(float("nan"))
        pr.barrier()                                              # everybody's inputs are in place
        pr.forward(sq, sk, sv, so, slse, softmax_scale=w.softmax_scale)
        pr.backward(sdo, sq, sk, sv, so, slse, sdq, sdk, sdv, ws, softmax_scale=w.softmax_scale)
        ok = True
        if rank == 0:
            plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
            cu = plan.cu_seqlens_dev("cuda")
            out, lse = sap.sap_attn_fwd(q, k, v, cu, plan, softmax_scale=w.softmax_scale)
            dq, dk, dv = sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale)
            torch.cuda.synchronize()
            assert torch.equal(sq, q) and torch.equal(sdo, do), "a peer's input rows are not visible"
            assert torch.equal(so, out) and torch.equal(slse, lse), "forward differs"
            assert torch.equal(sdk, dk) and torch.equal(sdv, dv), "dK / dV differ"
            check_close(to_np(sdq), to_np(dq), "dq, two processes vs single launch")
        pr.barrier()                                              # nobody unmaps while rank 0 still reads
        result_q.put((rank, ok))
    finally:
        dist.destroy_process_group()


def test_two_processes_share_stitched_tensors():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    try:
        res = sorted(q.get(timeout=240) for _ in procs)
    finally:
        for p in procs:
            p.join(30)
            if p.is_alive():
                p.kill()
    assert res == [(0, True), (1, True)]
    assert all(p.exitcode == 0 for p in procs)
