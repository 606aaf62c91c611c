"""Writes tests/golden/cu_seqlens_cfg{1..5}.txt from the seeded workload generator.

Calls only paper_2606_30460_b200.workloads (no oracle, no CUDA path).  Each file: the
document lengths, N, pairs = sum L(L+1)/2 and the SHA-256 of the cu_seqlens list; the tests
re-derive all of it so a drift of the generator is caught.
Run:  python tests/golden/make_cu_fixtures.py
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from paper_2606_30460_b200 import workloads as W  # noqa: E402

for cfg in range(1, 6):
    w = W.make_workload(cfg)
    with open(os.path.join(HERE, f"cu_seqlens_cfg{cfg}.txt"), "w") as f:
        f.write(f"# {w.name}: BASELINE.json configs[{cfg - 1}], seed 0 (recipe: workloads.py / DESIGN.md)\n")
        f.write(f"n_tokens {w.n_tokens}\nn_chunks {w.n_chunks}\nn_docs {len(w.doc_lens)}\n")
        f.write(f"pairs {w.pairs}\nsha256 {w.sha256()}\n")
        f.write("docs " + " ".join(map(str, w.doc_lens)) + "\n")
