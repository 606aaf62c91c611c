#!/usr/bin/env python
"""bench.py — useful causal TFLOP/s, fwd+bwd, of the SAP attention hot path on packed sequences.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A step = one pass of the whole hot path (plan already compiled ahead): sap_attn_fwd
(a2-a4) + sap_attn_bwd (a5-a7) over one seeded synthetic packed sequence of BASELINE.json configs[2]
(128K tokens, log-normal documents, 16 chunks, 32/8 heads, d=128) — the configuration the metric is
quoted on.  One JSON line on stdout (rank 0).  Multi-GPU: one process per GPU (`--gpus N` without a torchrun
environment starts the N ranks itself), no collective on the data path, two splits:
  --shard seqs  (default) independent packed sequences per rank, seed = rank: weak scaling;
  --shard heads one sequence, its kv-heads (with their q-heads) split over the ranks (heads are independent,
                PAPER.md:65): zero exchange, strong scaling.
`--dry-run` runs the host side only (planner, sharding, aggregation over gloo): no GPU needed.

`--impl reference` times the fp64 CPU oracle (oracle/), as it stands, on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "useful causal TFLOP/s fwd+bwd on packed seqs"
UNIT = "TFLOP/s"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"bf16_burst": p["bf16_tflops"], "bf16_sustained": p["bf16_tflops_sustained"],
                "hbm": p["hbm_gbs"], "source": "measured (MEASURED_PEAKS.json)"}
    return {"bf16_burst": 1590.0, "bf16_sustained": 1400.0, "hbm": 6650.0, "source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx = float(f[1])
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


ORACLE_SAMPLE_TOKENS = 2048   # the ONE sample both arms time the oracle on (about 6 s on 16 host threads)


def cpu_sample_workload(n_tokens: int):
    """Bounded sample of configs[2] for the oracle: its leading documents, cut at n_tokens, all heads."""
    from paper_2606_30460_b200.workloads import custom_workload, make_workload
    w3 = make_workload(3)
    lens, acc = [], 0
    for L in w3.doc_lens:
        L = min(L, n_tokens - acc)
        lens.append(L); acc += L
        if acc >= n_tokens:
            break
    return custom_workload(lens, 1, w3.n_q_heads, w3.n_kv_heads, w3.head_dim, name=f"cfg3_prefix_{n_tokens}")


def time_oracle(w, what: str):
    """fwd + dQ + dK/dV of the oracle, as it stands, on workload w; returns (seconds, useful flops, threads, description)."""
    from oracle import oracle
    from paper_2606_30460_b200.workloads import make_qkv
    q, k, v, do = (t.float().numpy() for t in make_qkv(w, device="cpu"))
    t0 = time.perf_counter()
    oracle.attn_fwd(q, k, v, w.cu_seqlens, w.softmax_scale)
    oracle.attn_bwd_dq(q, k, v, do, w.cu_seqlens, w.softmax_scale)
    oracle.attn_bwd_dkv(q, k, v, do, w.cu_seqlens, w.softmax_scale)
    dt = time.perf_counter() - t0
    desc = (f"{what} (docs {list(w.doc_lens)}), {w.n_q_heads}/{w.n_kv_heads} heads, d={w.head_dim}: oracle fwd + dQ + dK/dV, "
            f"every element")
    return dt, w.flops_fwd + w.flops_bwd, oracle.num_threads(), desc


def time_oracle_sample():
    return time_oracle(cpu_sample_workload(ORACLE_SAMPLE_TOKENS), f"first {ORACLE_SAMPLE_TOKENS} tokens of configs[2]")


def time_oracle_cfg1():
    from paper_2606_30460_b200.workloads import make_workload
    return time_oracle(make_workload(1), "configs[0] in full")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    for _ in range(args.warmup):
        time_oracle(cpu_sample_workload(256), "warm-up")
    tot_t, tot_f, threads, desc = 0.0, 0, 0, ""
    for _ in range(args.steps):
        dt, fl, threads, desc = time_oracle_sample()       # every step = the same fixed sample the GPU arm's cpu_baseline uses
        tot_t += dt; tot_f += fl
    val = tot_f / tot_t / 1e12
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot_t / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[2] 128K packed (bounded sample per step)", "sample": desc},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


PAPER_TABLE2_SAP_MS = {8192: 7.9, 16384: 11.1, 32768: 73.0, 65536: 1912.3, 131072: 3333.1}   # PAPER.md:158-164 (A100s, multi-GPU)


def table2_context(dev, steps: int = 5):
    """fwd+bwd time of one attention on the paper's Table 2 shape (16 heads MHA, d = 128, chunks =
    SP size; the paper's length mix is not stated, the recipe of configs[2] stands in), beside the paper's own SAP
    figure for that column - other hardware, transport included there: context, not a comparison."""
    import torch
    import paper_2606_30460_b200 as sap
    from paper_2606_30460_b200.workloads import make_qkv, make_table2_workload
    res = {}
    for L in (8192, 32768, 131072):
        w = make_table2_workload(L)
        q, k, v, do = make_qkv(w, device=dev)
        plan = sap.sap_plan(w.cu_seqlens, w.n_chunks); plan.upload()
        cu = plan.cu_seqlens_dev(dev)
        out = torch.empty_like(q); lse = torch.empty((w.n_q_heads, L), dtype=torch.float32, device=dev)
        dq, dk, dv = torch.empty_like(q), torch.empty_like(k), torch.empty_like(v)
        ws = torch.empty(sap.sap_workspace_bytes(plan, w.n_q_heads, w.n_kv_heads, w.head_dim, sap.SAP_PASS_BWD), dtype=torch.uint8, device=dev)

        def step():
            sap.sap_attn_fwd(q, k, v, cu, plan, out, lse, softmax_scale=w.softmax_scale)
            sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale, dq=dq, dk=dk, dv=dv, workspace=ws)

        for _ in range(3):
            step()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); e0.record()
        for _ in range(steps):
            step()
        e1.record(); torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        res[f"{L // 1024}K/SP{w.n_chunks}"] = {"ms_fwd_bwd": ms, "tflops": (w.flops_fwd + w.flops_bwd) / (ms * 1e-3) / 1e12,
                                               "n_docs": len(w.doc_lens), "paper_sap_ms_a100_multi_gpu": PAPER_TABLE2_SAP_MS[L]}
        del q, k, v, do, out, lse, dq, dk, dv, ws
    return res


def d64_context(dev, steps: int = 3):
    """SURVEY 8(f) NEXT-4, head_dim 64: configs[2]'s packing with 64 q-heads / 16 kv-heads of 64 (the same bytes per token),
    forward and backward timed apart.  At d = 64 a score costs half the tensor work but the same exponential: the
    forward keeps the MUFU (16 exp / clk / SM) over 80 % busy and cannot reach the d = 128 rate."""
    import torch
    import paper_2606_30460_b200 as sap
    from paper_2606_30460_b200.workloads import make_d64_workload, make_qkv
    w = make_d64_workload()     # parity at this size: tests/test_gpu_configs.py::test_d64_context_workload_sampled_against_oracle
    q, k, v, do = make_qkv(w, device=dev)
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks); plan.upload()
    cu = plan.cu_seqlens_dev(dev)
    out = torch.empty_like(q); lse = torch.empty((w.n_q_heads, w.n_tokens), dtype=torch.float32, device=dev)
    dq, dk, dv = torch.empty_like(q), torch.empty_like(k), torch.empty_like(v)
    ws = torch.empty(sap.sap_workspace_bytes(plan, w.n_q_heads, w.n_kv_heads, w.head_dim, sap.SAP_PASS_BWD), dtype=torch.uint8, device=dev)
    fns = {"fwd": lambda: sap.sap_attn_fwd(q, k, v, cu, plan, out, lse, softmax_scale=w.softmax_scale),
           "bwd": lambda: sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale, dq=dq, dk=dk, dv=dv, workspace=ws)}
    res = {"workload": w.name}
    for name, fn in fns.items():
        for _ in range(3):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); e0.record()
        for _ in range(steps):
            fn()
        e1.record(); torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        fl = w.flops_fwd if name == "fwd" else w.flops_bwd
        res[name] = {"ms": ms, "tflops": fl / (ms * 1e-3) / 1e12}
    return res


def kernel_source_sha256():
    """Hash of every source file that goes into libsap_b200.so: the key of profiles/traffic.json."""
    import hashlib
    root = os.path.join(ROOT, "paper_2606_30460_b200", "csrc")
    h = hashlib.sha256()
    for f in sorted(os.listdir(root)):
        h.update(f.encode()); h.update(open(os.path.join(root, f), "rb").read())
    return h.hexdigest()


def recorded_traffic(cfg: int, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` on BASELINE.json configs[cfg-1], from the
    committed ncu summary profiles/traffic.json - only if that capture was taken on this very kernel source."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(path):
        return None, None
    rec = json.load(open(path))
    if rec.get("kernel_source_sha256") != kernel_source_sha256():
        return None, "profiles/traffic.json was captured on another kernel source (hash differs): not reported"
    val = rec.get("bytes_per_launch", {}).get(f"cfg{cfg}", {}).get(kernel)
    return val, (rec.get("source") if val is not None else None)


def spawn_ranks(args):
    """`--gpus N` outside torchrun: start the N ranks (one process per GPU) under torch.distributed.run."""
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def run_dry(args):
    """Host side only (no GPU): sharding, planner and the aggregation collectives over gloo."""
    import torch.distributed as dist
    from paper_2606_30460_b200 import shard
    import paper_2606_30460_b200 as sap
    rank, world, _ = shard.rank_world()
    if world > 1:
        dist.init_process_group("gloo")
    extra = {}
    if args.shard == "chunks":       # one sequence, every head, rank r launches the chunks ranks.launch_chunks gives it
        from paper_2606_30460_b200.ranks import assign_by_work, chunk_work
        w = shard.rank_workload(args.config, 0)
        heads, share = tuple(range(w.n_kv_heads)), 1.0 / world
        q_work, kv_work = chunk_work(w.cu_seqlens, w.n_chunks)
        fwd_a, bwd_a = assign_by_work(q_work, world), assign_by_work(kv_work, world)
        extra = {"q_chunks_launched_by_rank": fwd_a, "kv_chunks_launched_by_rank": bwd_a,
                 "max_over_mean_load": {"fwd": max(sum(q_work[c] for c in x) for x in fwd_a) * world / sum(q_work),
                                        "bwd": max(sum(kv_work[c] for c in x) for x in bwd_a) * world / sum(kv_work)}}
    else:
        w, heads = shard.rank_share(args.config, rank, world, args.shard)
        share = len(heads) / w.n_kv_heads
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    ms_max, flops_all = shard.aggregate(1.0 + rank, float(w.flops_fwd + w.flops_bwd) * share)
    if rank == 0:
        print(json.dumps({"dry_run": True, "metric": METRIC, "n_gpus": world, "shard": args.shard, **extra,
                          "scaling": "weak" if args.shard == "seqs" else "strong", "plan_items": plan.n_items,
                          "kv_heads_of_rank0": list(heads), "whole_job_tflop_per_step": flops_all / 1e12,
                          "max_over_ranks_check": ms_max == float(world),
                          "config": {"workload": w.name, "n_tokens": w.n_tokens}}), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def run_chunks(args):
    """`--shard chunks`: the paper's sequence parallelism itself.  ONE packed sequence; rank r owns the
    memory of a contiguous block of its chunks (stitched tensors: ranks.ProcessRank) and launches the library's kernels on
    the chunks a work-balanced assignment gives it (visible pairs per chunk, from cu_seqlens); K/V, Q/dO and the dQ contributions travel inside the kernels (TMA and
    red.global over NVLink), the only synchronisation is four group barriers per step.  Strong scaling.  A step also
    includes, under `e2e`, every rank's own rows going host -> device and its results coming back."""
    import torch
    import torch.distributed as dist
    import paper_2606_30460_b200 as sap
    from paper_2606_30460_b200 import shard
    from paper_2606_30460_b200.ranks import ProcessRank
    from paper_2606_30460_b200.workloads import make_qkv

    rank, world, local = shard.rank_world()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    w = shard.rank_workload(args.config, 0)                     # the same sequence on every rank
    if w.n_chunks % world != 0:
        raise ValueError(f"--shard chunks needs n_chunks ({w.n_chunks}) divisible by the number of ranks ({world})")
    N, Hq, Hkv, d = w.n_tokens, w.n_q_heads, w.n_kv_heads, w.head_dim
    pr = ProcessRank(w.cu_seqlens, rank, world, device=local, n_chunks=w.n_chunks)
    q, do, out, dq = (pr.tensor((Hq, d), torch.bfloat16) for _ in range(4))
    k, v, dk, dv = (pr.tensor((Hkv, d), torch.bfloat16) for _ in range(4))
    lse = pr.shared((Hq, N), torch.float32)
    ws = pr.workspace(Hq, Hkv, d)
    rows = pr.own_rows()
    src = make_qkv(w, device=dev)                               # seeded: every rank can generate it, keeps its own rows
    host_in = [t[rows].cpu().pin_memory() for t in src]
    for dst, t in zip((q, k, v, do), src):
        dst[rows].copy_(t[rows])
    del src
    host_out = [torch.empty_like(t[rows], device="cpu").pin_memory() for t in (out, dq, dk, dv)]
    pr.barrier()

    def step():
        pr.forward(q, k, v, out, lse, softmax_scale=w.softmax_scale)
        pr.backward(do, q, k, v, out, lse, dq, dk, dv, ws, softmax_scale=w.softmax_scale)

    def step_e2e():
        for dst, t in zip((q, k, v, do), host_in):
            dst[rows].copy_(t, non_blocking=True)
        pr.barrier()                                            # everybody's inputs of this step are in place
        step()
        for dst, t in zip(host_out, (out, dq, dk, dv)):
            dst.copy_(t[rows], non_blocking=True)
        torch.cuda.synchronize()

    def timed(fn, n):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        pr.barrier()
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n

    for _ in range(max(args.warmup, 3)):
        step()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = sap.sap_launch_count()
    ms = timed(step, args.steps)
    launches = sap.sap_launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    flops = float(w.flops_fwd + w.flops_bwd)
    ms_max, flops_all = shard.aggregate(ms, flops / world, dev)
    ms_e2e = timed(step_e2e, max(3, min(args.steps, 10)))
    ms_e2e_max, _ = shard.aggregate(ms_e2e, 0.0, dev)
    if rank == 0:
        peaks = load_peaks()
        value = flops_all / (ms_max * 1e-3) / 1e12
        h2d = sum(t.numel() * t.element_size() for t in host_in) * world
        d2h = sum(t.numel() * t.element_size() for t in host_out) * world
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_max, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "bf16",
            "data": "synthetic",
            "config": {"workload": w.name, "n_tokens": N, "n_docs": len(w.doc_lens), "n_chunks": w.n_chunks, "n_q_heads": Hq,
                       "n_kv_heads": Hkv, "head_dim": d, "cu_seqlens_sha256": w.sha256(), "shard": "chunks",
                       "per_rank": "one sequence; rank 0 owns the memory of chunks %s and launches q-chunks %s / kv-chunks %s (balanced by "
                                   "visible pairs); stitched tensors, 4 group barriers per step, no collective on the data path"
                                   % (pr.owned, pr.launch, pr.launch_kv),
                       "l2": "inputs exceed L2"},
            "frac_of_bf16_peak": {"measured_burst": value / world / peaks["bf16_burst"],
                                  "measured_sustained": value / world / peaks["bf16_sustained"], "source": peaks["source"]},
            "clocks": clocks, "gpu_launches": launches * world,
            "e2e": {"value": flops_all / (ms_e2e_max * 1e-3) / 1e12, "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e_max,
                    "pipeline": "every rank copies its own rows in and its own results out, not overlapped"},
            "roofline": None, "cpu_baseline": None}), flush=True)
    pr.barrier()
    if world > 1:
        dist.destroy_process_group()


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2606_30460_b200 as sap
    from paper_2606_30460_b200 import shard
    from paper_2606_30460_b200.workloads import make_qkv

    rank, world, local = shard.rank_world()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # --shard seqs: each rank gets its own packed sequence (seed = rank): data-parallel units, no exchange;
    # --shard heads: one sequence, rank r keeps kv-heads `heads` and their q-heads (heads are independent)
    w, heads = shard.rank_share(args.config, rank, world, args.shard)
    q, k, v, do = make_qkv(w, device=dev)
    g = w.n_q_heads // w.n_kv_heads
    if len(heads) != w.n_kv_heads:
        qsel = [hk * g + i for hk in heads for i in range(g)]
        q, do = q[:, qsel].contiguous(), do[:, qsel].contiguous()
        k, v = k[:, list(heads)].contiguous(), v[:, list(heads)].contiguous()
    share = len(heads) / w.n_kv_heads
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    plan.upload()
    cu = plan.cu_seqlens_dev(dev)
    N, Hq, Hkv, d = w.n_tokens, q.shape[1], k.shape[1], w.head_dim
    out = torch.empty_like(q); lse = torch.empty((Hq, N), dtype=torch.float32, device=dev)
    dq, dk, dv = torch.empty_like(q), torch.empty_like(k), torch.empty_like(v)
    ws = torch.empty(sap.sap_workspace_bytes(plan, Hq, Hkv, d, sap.SAP_PASS_BWD), dtype=torch.uint8, device=dev)

    def fwd():
        sap.sap_attn_fwd(q, k, v, cu, plan, out, lse, softmax_scale=w.softmax_scale)

    def bwd():
        sap.sap_attn_bwd(do, q, k, v, out, lse, cu, plan, softmax_scale=w.softmax_scale, dq=dq, dk=dk, dv=dv, workspace=ws)

    def step():
        fwd(); bwd()

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed(fn, n):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n  # ms per call

    bwd_mask = 7 if args.bwd == "split" else -1   # -1 = library default (D pre-pass + fused main + dQ post pass)
    sap.sap_debug_set_bwd_stages(bwd_mask)
    sap.sap_debug_set_fwd_form(1 if args.fwd == "single" else 0)
    for _ in range(max(args.warmup, 3)):
        step()
    sync_all()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = sap.sap_launch_count()
    if args.graph:   # launch-bound shapes: the whole step captured once (no call allocates or synchronises), replayed K times
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            with torch.cuda.graph(graph, stream=side):
                step()
        per_step = sap.sap_launch_count() - launches0
        torch.cuda.current_stream().wait_stream(side)
        graph.replay(); torch.cuda.synchronize()
        ms = timed(graph.replay, args.steps)
        launches = per_step * args.steps
    else:
        ms = timed(step, args.steps)
        launches = sap.sap_launch_count() - launches0
    sync_all()
    clocks = sampler.stop() if rank == 0 else None
    ms_max, flops_all = shard.aggregate(ms, float(w.flops_fwd + w.flops_bwd) * share, dev)   # MAX time, SUM work
    value = flops_all / (ms_max * 1e-3) / 1e12

    # ---- per-kernel times (separate passes; CUDA events on the launching stream), rank 0 reports
    kn = max(3, min(args.steps, 10))
    t_fwd = timed(fwd, kn)
    per = {}
    if args.bwd == "split":
        for name, mask in (("bwd_pre", 1), ("bwd_dkv", 2), ("bwd_dq", 4)):
            sap.sap_debug_set_bwd_stages(mask)
            bwd(); torch.cuda.synchronize()
            per[name] = timed(bwd, kn)
        sap.sap_debug_set_bwd_stages(bwd_mask)
    else:   # the three phases of sap_attn_bwd through their own entry points (the per-rank calls over all chunks)
        P = w.n_chunks
        phases = {"bwd_pre": lambda: sap.sap_attn_bwd_begin(do, out, plan, 0, P, Hkv, ws),
                  "bwd_fused": lambda: sap.sap_attn_bwd_chunks(do, q, k, v, lse, cu, plan, 0, P, dk, dv, ws, softmax_scale=w.softmax_scale),
                  "bwd_post": lambda: sap.sap_attn_bwd_end(plan, 0, P, dq, Hkv, ws, softmax_scale=w.softmax_scale)}
        for name, fn in phases.items():
            fn(); torch.cuda.synchronize()
            per[name] = timed(fn, kn)
    main_kernel = "sap_bwd_pair_kernel" if d == 128 else "sap_bwd_fused_kernel"

    # ---- end to end: host (pinned) buffers in, results back to host, copies inside the timed region
    if args.profile_only:
        if world > 1:
            dist.destroy_process_group()
        if rank == 0:
            bwd_ms = sum(per.values())
            print(json.dumps({"profile_only": True, "workload": w.name, "n_tokens": N, "n_docs": len(w.doc_lens),
                              "useful_pairs": w.pairs, "plan_items": plan.n_items, "cu_seqlens_sha256": w.sha256(), "shard": args.shard, "n_gpus": world,
                              "bwd": args.bwd, "cuda_graph": bool(args.graph), "ms_per_step": ms_max, "value": value,
                              "frac_of_measured_burst_peak": value / world / load_peaks()["bf16_burst"],
                              "tokens_per_s": N * world / (ms_max * 1e-3), "fwd_ms": t_fwd,
                              "fwd_tflops": w.flops_fwd * share / (t_fwd * 1e-3) / 1e12, "bwd_ms": bwd_ms,
                              "bwd_tflops": w.flops_bwd * share / (bwd_ms * 1e-3) / 1e12, **per, "clocks": clocks}))
        return
    hq, hk, hv, hdo = (x.cpu().pin_memory() for x in (q, k, v, do))
    r_out, r_lse = torch.empty_like(hq).pin_memory(), torch.empty((Hq, N), dtype=torch.float32).pin_memory()
    r_dq, r_dk, r_dv = torch.empty_like(hq).pin_memory(), torch.empty_like(hk).pin_memory(), torch.empty_like(hv).pin_memory()

    # Double-buffered, three streams (a user's input pipeline): step i+1's inputs travel host -> device and step
    # i-1's results device -> host while step i computes.  Every step still copies its own inputs from pinned host
    # memory and reads its own results back; pipeline fill and drain are inside the timed region.
    s_comp, s_h2d, s_d2h = torch.cuda.current_stream(), torch.cuda.Stream(), torch.cuda.Stream()
    d_in = [(q, k, v, do), tuple(torch.empty_like(x) for x in (q, k, v, do))]
    d_out = [(out, lse, dq, dk, dv), tuple(torch.empty_like(x) for x in (out, lse, dq, dk, dv))]

    def e2e_run(n):
        qkv_ready = [torch.cuda.Event() for _ in range(n)]
        do_ready = [torch.cuda.Event() for _ in range(n)]
        fwd_done = [torch.cuda.Event() for _ in range(n)]
        comp_done = [torch.cuda.Event() for _ in range(n)]
        d2h_done = [torch.cuda.Event() for _ in range(n)]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(s_h2d)
        for i in range(n):
            sl = i & 1
            qi, ki, vi, doi = d_in[sl]
            oi, li, dqi, dki, dvi = d_out[sl]
            with torch.cuda.stream(s_h2d):
                if i >= 2:
                    s_h2d.wait_event(comp_done[i - 2])          # the slot's inputs have been consumed
                for dst, src in zip((qi, ki, vi), (hq, hk, hv)):
                    dst.copy_(src, non_blocking=True)
                qkv_ready[i].record(s_h2d)                      # the forward needs only Q, K, V ...
                doi.copy_(hdo, non_blocking=True)
                do_ready[i].record(s_h2d)                       # ... dO travels under it
            s_comp.wait_event(qkv_ready[i])
            if i >= 2:
                s_comp.wait_event(d2h_done[i - 2])              # the slot's previous results have been read back
            sap.sap_attn_fwd(qi, ki, vi, cu, plan, oi, li, softmax_scale=w.softmax_scale)
            fwd_done[i].record(s_comp)
            s_comp.wait_event(do_ready[i])
            sap.sap_attn_bwd(doi, qi, ki, vi, oi, li, cu, plan, softmax_scale=w.softmax_scale, dq=dqi, dk=dki, dv=dvi,
                             workspace=ws)
            comp_done[i].record(s_comp)
            with torch.cuda.stream(s_d2h):
                s_d2h.wait_event(fwd_done[i])                   # out and LSE go back while the backward runs
                r_out.copy_(oi, non_blocking=True); r_lse.copy_(li, non_blocking=True)
                s_d2h.wait_event(comp_done[i])
                for dst, src in zip((r_dq, r_dk, r_dv), (dqi, dki, dvi)):
                    dst.copy_(src, non_blocking=True)
                d2h_done[i].record(s_d2h)
        e1.record(s_d2h)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n

    e2e_run(2); sync_all()
    e_steps = max(4, min(args.steps, 32))   # pipeline fill and drain are inside the timed region: the same K as the main loop
    ms_e2e = e2e_run(e_steps)
    sync_all()
    ms_e2e_max, _ = shard.aggregate(ms_e2e, 0.0, dev)
    e2e_value = flops_all / (ms_e2e_max * 1e-3) / 1e12
    h2d = sum(x.numel() * x.element_size() for x in (hq, hk, hv, hdo))
    d2h = sum(x.numel() * x.element_size() for x in (r_out, r_lse, r_dq, r_dk, r_dv))

    if rank == 0:
        peaks = load_peaks()
        pairs = w.pairs
        # algorithmic FLOPs per launch: 2*d flops per visible (row, key) pair per
        # q-head per GEMM; fwd = 2 GEMMs, dK/dV kernel = 4 of the backward's 5 (S, dP, dV, dK), dQ kernel = 1 (dQ;
        # its S/dP recompute is overhead, not algorithmic work)
        gemm = 2.0 * d * Hq * pairs       # Hq = this rank's q-heads
        kernels = {
            "sap_fwd_kernel": {"ms": t_fwd, "algorithmic_tflop": 2 * gemm / 1e12},
            "sap_bwd_pre_kernel": {"ms": per["bwd_pre"], "algorithmic_gbytes": (2 * N * Hq * d * 2 + N * Hq * 4) / 1e9},
        }
        if args.bwd == "split":
            kernels["sap_bwd_dkv_kernel"] = {"ms": per["bwd_dkv"], "algorithmic_tflop": 4 * gemm / 1e12}
            kernels["sap_bwd_dq_kernel"] = {"ms": per["bwd_dq"], "algorithmic_tflop": 1 * gemm / 1e12,
                                            "executed_tflop": 3 * gemm / 1e12}
        else:
            # main kernel: all 5 GEMMs of the backward (the D pre-pass line includes zeroing the fp32 dQ accumulator)
            kernels[main_kernel] = {"ms": per["bwd_fused"], "algorithmic_tflop": 5 * gemm / 1e12}
            # sap_attn_bwd_begin = D pre-pass + cudaMemsetAsync of the fp32 dQ accumulator: count the zeroed bytes too
            kernels["sap_bwd_pre_kernel"]["algorithmic_gbytes"] += N * Hq * d * 4 / 1e9
            kernels["sap_bwd_pre_kernel"]["includes"] = "cudaMemsetAsync of the fp32 dQ accumulator"
            kernels["sap_bwd_post_kernel"] = {"ms": per["bwd_post"], "algorithmic_gbytes": N * Hq * d * 6 / 1e9}
        for kk, vv in kernels.items():
            if "algorithmic_tflop" in vv:
                vv["tflops"] = vv["algorithmic_tflop"] / (vv["ms"] * 1e-3)
                vv["frac_of_bf16_burst"] = vv["tflops"] / peaks["bf16_burst"]
            else:
                vv["gbs"] = vv["algorithmic_gbytes"] / (vv["ms"] * 1e-3)
                vv["frac_of_hbm"] = vv["gbs"] / peaks["hbm"]
        dom = max((kk for kk in kernels if "tflops" in kernels[kk]), key=lambda kk: kernels[kk]["ms"])
        # DRAM bytes per launch of the dominant kernel from the committed `ncu --set full` summary, if it was taken
        # on this kernel source and this configuration (null otherwise)
        traffic, traffic_src = recorded_traffic(args.config, dom) if (world == 1 and args.shard == "seqs") else (None, None)
        roofline = {"kernel": dom, "bound": "tensor", "achieved": kernels[dom]["tflops"],
                    "peak": peaks["bf16_sustained"], "unit": "TFLOP/s",
                    "frac": kernels[dom]["tflops"] / peaks["bf16_sustained"], "traffic": traffic,
                    "peak_source": peaks["source"] + ", sustained bf16 (kernel timed inside a long step)",
                    "ms_per_launch": kernels[dom]["ms"],
                    "traffic_source": traffic_src}
        t2 = table2_context(dev) if (world == 1 and args.config == 3) else None
        d64 = d64_context(dev) if (world == 1 and args.config == 3) else None
        cdt, cfl, cthreads, cdesc = time_oracle_sample()
        c1dt, c1fl, _, c1desc = time_oracle_cfg1()
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_max, "higher_is_better": True,
            "scaling": "strong" if args.shard == "heads" else "weak",
            "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": (f"BASELINE.json configs[{args.config - 1}]: {w.name}" if args.config <= 5 else
                                    f"head_dim 64 context (not a BASELINE config): {w.name}" if args.config == 64 else
                                    f"paper Table 2 shape (context, not a BASELINE config): {w.name}"), "n_tokens": N,
                       "n_chunks": w.n_chunks, "n_docs": len(w.doc_lens), "n_q_heads": Hq, "n_kv_heads": Hkv,
                       "head_dim": d, "cu_seqlens_sha256": w.sha256(), "useful_pairs": pairs,
                       "plan_items": plan.n_items, "l2": "inputs exceed L2 (Q alone is %.0f MiB)" % (q.numel() * 2 / 2**20),
                       "per_rank": ("independent sequence per rank (seed = rank)" if args.shard == "seqs" else
                                    f"one sequence, {Hkv} of its {w.n_kv_heads} kv-heads (and their q-heads) per rank, no exchange"),
                       "shard": args.shard, "bwd": args.bwd, "cuda_graph": bool(args.graph)},
            "tokens_per_s": N * world / (ms_max * 1e-3),
            "frac_of_bf16_peak": {"measured_burst": value / world / peaks["bf16_burst"],
                                  "measured_sustained": value / world / peaks["bf16_sustained"],
                                  "datasheet_2250": value / world / 2250.0, "source": peaks["source"]},
            "fwd": {"ms": t_fwd, "tflops": w.flops_fwd * share / (t_fwd * 1e-3) / 1e12},
            "bwd": {"ms": sum(per.values()), "tflops": w.flops_bwd * share / (sum(per.values()) * 1e-3) / 1e12},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": ms_e2e_max, "steps": e_steps,
                    "pipeline": "double-buffered, 3 streams: H2D of step i+1 and D2H of step i-1 overlap step i; dO travels under the forward, out / LSE go back under the backward"},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "kernels": kernels,
            "cpu_baseline": {"value": cfl / cdt / 1e12, "unit": UNIT, "cores": cthreads, "kind": "oracle",
                             "sample": cdesc, "seconds": cdt,
                             # not run: the sample's rate applied to the whole workload's useful FLOPs (the oracle's cost per
                             # visible pair does not depend on the document it lies in)
                             "extrapolated": {"full_config_seconds": (w.flops_fwd + w.flops_bwd) / (cfl / cdt),
                                              "label": "extrapolated from the sample's rate, not measured"},
                             "cfg1_full": {"value": c1fl / c1dt / 1e12, "unit": UNIT, "seconds": c1dt, "sample": c1desc}},
            "table2_context": t2, "d64_context": d64,
            "paper_context": "HSAP Table 2 (PAPER.md:158-164): SAP attention fwd+bwd 128K/SP16 = 3333.1 ms on A100s, "
                             "multi-GPU, communication included; not comparable, context only",
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="1..5 = BASELINE.json configs[0..4]; 64 = head_dim 64 on configs[2]'s packing (context); 8192..131072 = the paper's Table 2 shape at that length (context)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--fwd", default="pair", choices=["pair", "single"],
                    help="forward kernel: two q-heads per CTA (default when Hq/Hkv is even) or one (diagnostic)")
    ap.add_argument("--bwd", default="fused", choices=["fused", "split"],
                    help="backward form: fused 5-GEMM kernel (default) or the split dK/dV + dQ kernels (diagnostic)")
    ap.add_argument("--shard", default="seqs", choices=["seqs", "heads", "chunks"],
                    help="multi-GPU split: independent sequences per rank (weak scaling), the kv-heads of one sequence (strong), or "
                         "the chunks of one sequence = the paper's sequence parallelism over stitched tensors (strong)")
    ap.add_argument("--graph", action="store_true", help="time replays of one captured CUDA graph of the step (launch-bound shapes)")
    ap.add_argument("--dry-run", action="store_true", help="host side only (planner, sharding, aggregation over gloo); no GPU")
    ap.add_argument("--profile-only", action="store_true",
                    help="stop after the device-timed region and the per-kernel passes (for ncu runs)")
    args = ap.parse_args()
    if args.gpus > 1 and "RANK" not in os.environ and args.impl == "ours":
        spawn_ranks(args)              # one process per GPU; this process only waits for them
    if args.impl == "reference":
        run_reference(args)
    elif args.dry_run:
        run_dry(args)
    elif args.shard == "chunks":
        run_chunks(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
