"""SAP ranks driven from ONE process over stitched tensors (the B200-native exchange).

The paper's ranks exchange K/V (and dK/dV, dQ) shards with grouped send / recv around a FlashAttention call
(PAPER.md:59, :100-102, :124).  Inside an NVLink / NVSwitch domain nothing has to be shipped ahead of the kernel: every
[N, H, d] tensor lives in one stitched range (`api.Stitched`: chunk c = memory of the device that owns sequence chunk
c), all tensors keep global token indices, and rank c launches the library's kernels restricted to its own chunks on
its own device.  Its forward reads the K/V tiles its plan names where they live (TMA over NVLink), its KV-stationary
backward streams Q / dO the same way and adds its dQ contributions into the owner's fp32 accumulator (red.global) -
transfer and compute are one kernel, and the chunk pairs the plan skips move no byte.

Control flow = four phases with two group barriers (stream events; no kernel ever waits on another kernel):
    forward:  every rank: sap_attn_fwd_chunks(own q-chunk)
    backward: every rank: sap_attn_bwd_begin(own rows: D, zeroed accumulator)   | barrier: all D written, all rows zeroed
              every rank: sap_attn_bwd_chunks(own K/V chunk)                     | barrier: all contributions added
              every rank: sap_attn_bwd_end(own dQ rows)
Ranks that share a device share its stream (their launches run one after the other): with every chunk on device 0 this
is the one-GPU emulation the tests run; with distinct P2P-capable devices it is the multi-GPU form - not run anywhere
yet (no box with a second GPU), so treat that path as untested.  One process drives all devices; the one-process-per-GPU
form needs the stitched handles exported between processes, which is not built.
"""
from __future__ import annotations

from typing import Dict, List, Optional, Sequence

from . import api


class RankGroup:
    def __init__(self, cu_seqlens: Sequence[int], n_chunks: int, devices: Optional[Sequence[int]] = None):
        import torch
        self.P = int(n_chunks)
        self.devices: List[int] = [0] * self.P if devices is None else [int(d) for d in devices]
        if len(self.devices) != self.P:
            raise ValueError("one device per chunk")
        self.cu_seqlens = list(cu_seqlens)
        self.n_tokens = int(self.cu_seqlens[-1])
        self.plans: Dict[int, api.Plan] = {}
        self.cu_dev = {}
        self.streams = {}
        for dev in sorted(set(self.devices)):          # a plan's device mirror lives on one device: one plan per device
            with torch.cuda.device(dev):
                plan = api.sap_plan(self.cu_seqlens, self.P)
                plan.upload()
                self.plans[dev] = plan
                self.cu_dev[dev] = plan.cu_seqlens_dev(torch.device("cuda", dev))
                self.streams[dev] = torch.cuda.Stream(device=dev)
        self._keep = []

    # ------------------------------------------------------------------ memory
    def tensor(self, tail_shape: Sequence[int], dtype):
        """[N, *tail_shape] in a stitched range: rows of chunk c in the memory of devices[c]."""
        import torch
        n = self.n_tokens // self.P
        row = 1
        for x in tail_shape:
            row *= int(x)
        chunk_bytes = n * row * torch.empty((), dtype=dtype).element_size()
        s = api.Stitched(self.P, chunk_bytes, self.devices, sorted(set(self.devices)))
        return s.tensor((self.n_tokens, *tail_shape), dtype)

    def shared(self, shape: Sequence[int], dtype):
        """An array every rank reads and writes rows of but that cannot be split by chunk ([Hq, N] LSE, the backward
        workspace): one allocation on the first device, mapped for all of them."""
        import torch
        nbytes = torch.empty((), dtype=dtype).element_size()
        for x in shape:
            nbytes *= int(x)
        g = api.Stitched.granularity(self.devices[0])
        s = api.Stitched(1, (nbytes + g - 1) // g * g, [self.devices[0]], sorted(set(self.devices)))
        return s.tensor(tuple(shape), dtype)

    def workspace(self, n_q_heads: int, n_kv_heads: int, head_dim: int):
        import torch
        plan = self.plans[self.devices[0]]
        return self.shared((api.sap_workspace_bytes(plan, n_q_heads, n_kv_heads, head_dim, api.SAP_PASS_BWD),), torch.uint8)

    # ------------------------------------------------------------------ control
    def _fork(self):
        import torch
        for dev, st in self.streams.items():
            ev = torch.cuda.Event()
            with torch.cuda.device(self.devices[0]):
                ev.record(torch.cuda.current_stream())
            st.wait_event(ev)

    def _barrier(self):
        """Every rank's stream waits for the work every other rank's stream has been given so far."""
        import torch
        evs = []
        for dev, st in self.streams.items():
            ev = torch.cuda.Event()
            ev.record(st)
            evs.append(ev)
        for st in self.streams.values():
            for ev in evs:
                st.wait_event(ev)

    def _join(self):
        import torch
        cur = torch.cuda.current_stream(self.devices[0])
        for st in self.streams.values():
            ev = torch.cuda.Event()
            ev.record(st)
            cur.wait_event(ev)

    def _each_rank(self, fn):
        import torch
        for c, dev in enumerate(self.devices):
            with torch.cuda.device(dev):
                fn(c, self.plans[dev], self.cu_dev[dev], self.streams[dev])

    def forward(self, q, k, v, out, lse, softmax_scale: Optional[float] = None):
        self._fork()
        self._each_rank(lambda c, plan, cu, st: api.sap_attn_fwd_chunks(q, k, v, cu, plan, c, c + 1, out, lse,
                                                                        softmax_scale=softmax_scale, stream=st))
        self._join()

    def backward(self, dout, q, k, v, out, lse, dq, dk, dv, workspace, softmax_scale: Optional[float] = None):
        n_kv_heads = k.shape[1]
        self._fork()
        self._each_rank(lambda c, plan, cu, st: api.sap_attn_bwd_begin(dout, out, plan, c, c + 1, n_kv_heads, workspace, stream=st))
        self._barrier()        # every D written, every accumulator row zeroed
        self._each_rank(lambda c, plan, cu, st: api.sap_attn_bwd_chunks(dout, q, k, v, lse, cu, plan, c, c + 1, dk, dv, workspace,
                                                                        softmax_scale=softmax_scale, stream=st))
        self._barrier()        # every dQ contribution added
        self._each_rank(lambda c, plan, cu, st: api.sap_attn_bwd_end(plan, c, c + 1, dq, n_kv_heads, workspace,
                                                                     softmax_scale=softmax_scale, stream=st))
        self._join()
