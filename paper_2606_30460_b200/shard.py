"""Data-parallel sharding of the hot path over ranks (one process per GPU).

The path partitions into independent problems (packed sequences), so ranks exchange nothing on the
data path: rank r works on its own seeded sequence and the only collectives are the ones that aggregate the
timing (MAX over ranks) and the work done (SUM over ranks).  Works on any torch.distributed backend (nccl on
GPUs, gloo in the CPU tests); with no initialised process group it degrades to the single-rank identity.
"""
from __future__ import annotations

import os
from typing import Tuple

from .workloads import Workload, make_d64_workload, make_table2_workload, make_workload


def rank_world() -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) from the torchrun environment (defaults: single process)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def rank_workload(cfg: int, rank: int) -> Workload:
    """The packed sequence rank `rank` works on: same recipe, seed = rank (weak scaling: fixed work per rank)."""
    if cfg == 64:        # head_dim 64 on configs[2]'s packing (context runs, NEXT-4)
        return make_d64_workload(seed=rank)
    if cfg > 5:          # 8192, 16384, ...: the paper's Table 2 shape at that length (context runs, NEXT-4)
        return make_table2_workload(cfg, seed=rank)
    return make_workload(cfg, seed=rank)


def rank_share(cfg: int, rank: int, world: int, how: str = "seqs"):
    """(workload, kv-heads) of rank `rank`.  how = "seqs": its own sequence (seed = rank), all heads (weak scaling);
    how = "heads": THE sequence (seed 0) and an equal contiguous share of its kv-heads - heads are independent
    (multi-head attention "as H independent single head attention"; IntraSP shards them, :65), so the
    ranks exchange nothing (strong scaling)."""
    if how == "seqs":
        w = rank_workload(cfg, rank)
        return w, tuple(range(w.n_kv_heads))
    w = rank_workload(cfg, 0)
    if w.n_kv_heads % world != 0:
        raise ValueError(f"--shard heads needs n_kv_heads ({w.n_kv_heads}) divisible by the number of ranks ({world})")
    per = w.n_kv_heads // world
    return w, tuple(range(rank * per, (rank + 1) * per))


def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def barrier() -> None:
    d = _dist()
    if d is not None:
        d.barrier()


def aggregate(ms: float, units: float, device="cpu") -> Tuple[float, float]:
    """(max over ranks of `ms`, sum over ranks of `units`): whole-job time and whole-job work of one step."""
    import torch
    d = _dist()
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    if d is not None:
        d.all_reduce(t, op=d.ReduceOp.MAX)
        d.all_reduce(u, op=d.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def throughput(ms: float, units: float, device="cpu") -> float:
    """Whole-job units per second: units all ranks processed / the slowest rank's time."""
    ms_max, units_all = aggregate(ms, units, device)
    return units_all / (ms_max * 1e-3)
