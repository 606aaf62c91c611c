"""Multi-rank host logic on CPU: world_size-2 `gloo` process group (no GPU).  The data path has no collective
(ranks own independent packed sequences); what is tested is the sharding recipe and the MAX / SUM aggregation
bench.py reports, plus that two ranks build different, valid plans."""
import os
import socket

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_30460_b200 import shard


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import paper_2606_30460_b200 as sap
        assert shard.rank_world() == (rank, world, rank)
        w = shard.rank_workload(2, rank)
        plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)          # host planner only: no GPU needed
        ms = 10.0 + 5.0 * rank                                   # rank 1 is the slow one
        units = float(w.flops_fwd + w.flops_bwd)
        shard.barrier()
        ms_max, units_all = shard.aggregate(ms, units)
        tput = shard.throughput(ms, units)
        q.put((rank, w.sha256(), w.n_tokens, plan.n_items, int(plan.useful_pairs), w.pairs, units, ms_max, units_all, tput))
    finally:
        dist.destroy_process_group()


def test_two_ranks_shard_and_aggregate():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    (r0, sha0, n0, items0, up0, pairs0, u0, mx0, ua0, t0), (r1, sha1, n1, items1, up1, pairs1, u1, mx1, ua1, t1) = res
    assert (r0, r1) == (0, 1)
    assert sha0 != sha1 and n0 == n1 == 32768            # different sequences, same size (weak scaling)
    assert up0 == pairs0 and up1 == pairs1 and items0 >= 8 and items1 >= 8
    assert mx0 == mx1 == 15.0                             # MAX over ranks
    assert ua0 == ua1 == u0 + u1                          # SUM over ranks
    assert np.isclose(t0, (u0 + u1) / 15e-3) and t0 == t1


def test_single_process_identity():
    assert shard.aggregate(3.0, 7.0) == (3.0, 7.0)
    assert shard.throughput(2.0, 10.0) == 5000.0
    assert shard.rank_workload(3, 0).sha256() == "15891bb89fd3d78b99a0e5215cd768c9a39887ff1d51582c827e62e545a073b4"
