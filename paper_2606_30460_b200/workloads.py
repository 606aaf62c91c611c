"""Seeded synthetic inputs for the SAP attention hot path.

This module holds NONE of the method's arithmetic: it only draws document
lengths and Q/K/V/dO values.  It is the one module both the CUDA path's tests /
bench and the oracle's tests may share (it imports neither of them).

The five configurations are BASELINE.json's `configs`; they stand in for the
paper's FineWeb / SlimPajama / UltraChat length mixes (§4.2),
which are not available here and whose histograms the paper does not print.
Recipe (also stated in DESIGN.md §Inputs):

  document length L = round(exp(ln(median) + sigma * z)), z ~ N(0,1),
  clipped to [lo, hi], appended until the total reaches N, last one truncated.
  z comes from a self-contained SplitMix64 + Box-Muller stream so the fixture
  lists under tests/golden/ do not depend on a numpy version.

  Q, K, V, dO ~ iid N(0,1) drawn in fp32 and rounded to bf16 (RNE), one
  torch.Generator per tensor seeded (seed*4 + index), on the device asked for.
"""
from __future__ import annotations

import hashlib
import math
from dataclasses import dataclass
from typing import List, Sequence

_MASK64 = (1 << 64) - 1


class SplitMix64:
    """Counter-based 64-bit generator (Steele, Lea, Flood 2014)."""

    def __init__(self, seed: int):
        self.state = seed & _MASK64

    def next_u64(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & _MASK64
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK64
        return z ^ (z >> 31)

    def uniform(self) -> float:
        """Uniform in (0, 1): 53 random bits, never exactly 0."""
        return ((self.next_u64() >> 11) + 0.5) / float(1 << 53)

    def normal(self) -> float:
        """One N(0,1) draw by Box-Muller (cosine branch only, two uniforms)."""
        u1 = self.uniform()
        u2 = self.uniform()
        return math.sqrt(-2.0 * math.log(u1)) * math.cos(2.0 * math.pi * u2)

    def randint(self, lo: int, hi: int) -> int:
        """Uniform integer in [lo, hi] (modulo bias < 2^-50, irrelevant here)."""
        return lo + self.next_u64() % (hi - lo + 1)


def lognormal_doc_lengths(rng: SplitMix64, total: int, median: float, sigma: float,
                          lo: int, hi: int) -> List[int]:
    """Log-normal lengths clipped to [lo, hi], appended until `total`; last truncated."""
    out: List[int] = []
    acc = 0
    while acc < total:
        L = int(round(math.exp(math.log(median) + sigma * rng.normal())))
        L = max(lo, min(hi, L))
        L = min(L, total - acc)
        out.append(L)
        acc += L
    return out


def uniform_doc_lengths(rng: SplitMix64, total: int, lo: int, hi: int) -> List[int]:
    out: List[int] = []
    acc = 0
    while acc < total:
        L = min(rng.randint(lo, hi), total - acc)
        out.append(L)
        acc += L
    return out


@dataclass(frozen=True)
class Workload:
    name: str
    n_tokens: int
    n_chunks: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    doc_lens: tuple
    seed: int = 0

    @property
    def cu_seqlens(self) -> List[int]:
        cu = [0]
        for L in self.doc_lens:
            cu.append(cu[-1] + L)
        return cu

    @property
    def softmax_scale(self) -> float:
        return 1.0 / math.sqrt(self.head_dim)

    @property
    def pairs(self) -> int:
        """Useful (row, key) pairs: sum over documents of L(L+1)/2 (exact integer)."""
        return sum(L * (L + 1) // 2 for L in self.doc_lens)

    @property
    def flops_fwd(self) -> int:
        """QK^T and PV: 2 GEMMs x 2 flops x d per pair per q-head."""
        return 4 * self.head_dim * self.n_q_heads * self.pairs

    @property
    def flops_bwd(self) -> int:
        """5 GEMMs (S recompute, dP, dV, dK, dQ): the usual 2.5x convention."""
        return 10 * self.head_dim * self.n_q_heads * self.pairs

    def sha256(self) -> str:
        return hashlib.sha256((" ".join(map(str, self.cu_seqlens))).encode()).hexdigest()


def make_workload(cfg: int, seed: int = 0) -> Workload:
    """cfg in 1..5 = BASELINE.json configs[0..4]."""
    rng = SplitMix64(0x5A9C0DE ^ (cfg * 1000003) ^ (seed * 7919))
    if cfg == 1:
        return Workload("cfg1_tiny_2k", 2048, 4, 4, 4, 64, (700, 1100, 248), seed)
    if cfg == 2:
        docs = lognormal_doc_lengths(rng, 32768, 2048, 1.0, 64, 32768)
        return Workload("cfg2_packed_32k", 32768, 8, 32, 8, 128, tuple(docs), seed)
    if cfg == 3:
        docs = lognormal_doc_lengths(rng, 131072, 4096, 1.2, 128, 131072)
        return Workload("cfg3_packed_128k", 131072, 16, 32, 8, 128, tuple(docs), seed)
    if cfg == 4:
        return Workload("cfg4_single_128k", 131072, 16, 32, 8, 128, (131072,), seed)
    if cfg == 5:
        n = 524288
        n_short = n // 5
        long_docs = lognormal_doc_lengths(rng, n - n_short, 8192, 1.5, 256, 262144)
        short_docs = uniform_doc_lengths(rng, n_short, 64, 512)
        docs = long_docs + short_docs
        for i in range(len(docs) - 1, 0, -1):          # Fisher-Yates: "interleaved"
            j = rng.randint(0, i)
            docs[i], docs[j] = docs[j], docs[i]
        return Workload("cfg5_packed_512k", n, 64, 32, 8, 128, tuple(docs), seed)
    raise ValueError(f"unknown config {cfg}")


# the shape of the paper's own attention micro-benchmark (Table 2, PAPER.md:158-164, :173:
# 16 heads MHA, "hidden_size" 128 read as head_dim, max sequence length 8K..128K, SP size = chunk count).  The paper
# does not state its "hybrid-context" length mix; the log-normal recipe of configs[2] scaled to the length stands in.
TABLE2_SP = {8192: 2, 16384: 4, 32768: 8, 65536: 16, 131072: 16}


def make_table2_workload(seq_len: int, seed: int = 0) -> Workload:
    if seq_len not in TABLE2_SP:
        raise ValueError(f"Table 2 lengths are {sorted(TABLE2_SP)}")
    rng = SplitMix64(0x7AB1E2 ^ (seq_len * 31) ^ (seed * 7919))
    docs = lognormal_doc_lengths(rng, seq_len, seq_len / 32, 1.2, 128, seq_len)
    return Workload(f"table2_{seq_len // 1024}k_sp{TABLE2_SP[seq_len]}", seq_len, TABLE2_SP[seq_len], 16, 16, 128,
                    tuple(docs), seed)


def make_d64_workload(seed: int = 0) -> Workload:
    """SURVEY 8(f) NEXT-4, head_dim 64: configs[2]'s packing with 64 q-heads on 16 kv-heads of 64 (the same bytes per
    token as configs[2]).  What bench.py's `d64_context` times and tests/test_gpu_configs.py checks."""
    w0 = make_workload(3, seed=seed)
    return custom_workload(w0.doc_lens, w0.n_chunks, 64, 16, 64, seed=w0.seed, name="configs[2] packing, 64/16 heads, d=64")


def custom_workload(doc_lens: Sequence[int], n_chunks: int, n_q_heads: int, n_kv_heads: int,
                    head_dim: int, seed: int = 0, name: str = "custom") -> Workload:
    return Workload(name, int(sum(doc_lens)), n_chunks, n_q_heads, n_kv_heads, head_dim,
                    tuple(int(x) for x in doc_lens), seed)


def make_qkv(w: Workload, device="cpu", with_dout: bool = True):
    """Q [N,Hq,d], K,V [N,Hkv,d], dO [N,Hq,d] in bf16 ~ N(0,1), seeded per tensor."""
    import torch

    def draw(idx: int, heads: int):
        g = torch.Generator(device=device)
        g.manual_seed(w.seed * 4 + idx + 1234)
        n_el = w.n_tokens * heads * w.head_dim
        out = torch.empty((w.n_tokens, heads, w.head_dim), dtype=torch.bfloat16, device=device)
        flat = out.view(-1)
        step = 1 << 26                                  # bounded fp32 staging
        for s in range(0, n_el, step):
            e = min(n_el, s + step)
            flat[s:e] = torch.randn(e - s, generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)
        return out

    q = draw(0, w.n_q_heads)
    k = draw(1, w.n_kv_heads)
    v = draw(2, w.n_kv_heads)
    if not with_dout:
        return q, k, v
    do = draw(3, w.n_q_heads)
    return q, k, v, do
