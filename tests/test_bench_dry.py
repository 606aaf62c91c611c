"""`bench.py --gpus N` starts its N ranks itself: run the host side of the bench (planner, sharding,
aggregation over gloo; no GPU) with two ranks, for both splits of SURVEY 8(e)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*extra):
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--dry-run", "--config", "2", *extra],
                         capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, out.stdout          # rank 0 alone prints
    return json.loads(lines[0])


@pytest.mark.parametrize("shard, scaling", [("seqs", "weak"), ("heads", "strong"), ("chunks", "strong")])
def test_bench_gpus_2_spawns_two_ranks(shard, scaling):
    one = run_bench("--shard", shard)
    two = run_bench("--gpus", "2", "--shard", shard)
    assert one["n_gpus"] == 1 and two["n_gpus"] == 2 and two["scaling"] == scaling
    assert two["max_over_ranks_check"] is True               # the MAX-over-ranks all-reduce saw both ranks
    if shard == "heads":                                     # one sequence split by kv-heads: the same total work
        assert two["kv_heads_of_rank0"] == [0, 1, 2, 3]
        assert two["whole_job_tflop_per_step"] == pytest.approx(one["whole_job_tflop_per_step"])
    elif shard == "chunks":                                  # one sequence split by chunks (the paper's SP): zig-zag launches
        for key in ("q_chunks_launched_by_rank", "kv_chunks_launched_by_rank"):      # a partition of the 8 chunks
            assert sorted(sum(two[key], [])) == list(range(8)) and len(two[key]) == 2
        assert two["max_over_mean_load"]["fwd"] < 1.1 and two["max_over_mean_load"]["bwd"] < 1.1
        assert two["whole_job_tflop_per_step"] == pytest.approx(one["whole_job_tflop_per_step"])
    else:                                                    # independent sequences: work adds up (different seeds)
        assert two["whole_job_tflop_per_step"] > one["whole_job_tflop_per_step"]
