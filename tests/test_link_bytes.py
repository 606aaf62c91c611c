"""ranks.link_bytes: the NVLink traffic of the two multi-GPU data planes, counted from the tile programs (host only).
Pinned by a case small enough to count by hand, by invariants, and printed for configs[2] / configs[4] at 2, 4, 8 ranks
(the table of DESIGN.md section 8 is this output)."""
import pytest

from paper_2606_30460_b200.ranks import chunk_work, link_bytes
from paper_2606_30460_b200.workloads import make_workload

KB = 1024


def test_one_document_two_ranks_by_hand():
    # 1024 tokens, one document, 2 chunks of 512 on 2 ranks, one head of 64.
    # forward, rank 1: its Q tiles at rows 512, 640, 768, 896 each stream the key tiles 0, 128, 256, 384 of rank 0:
    #   16 remote tile loads of K + V = 2 * 128 * 64 * 2 B = 32 KB each
    # backward, rank 0: its K/V tiles 0..384 each stream the row tiles 512..896 of rank 1: 16 remote (tile, tile) pairs of
    #   Q + dO (32 KB) + LSE + D (1 KB) read and 128 * 64 * 4 B = 32 KB of dQ contributions sent
    st = link_bytes([0, 1024], 2, 2, "stitched", 1, 1, 64)
    assert st == [{"fwd_read": 0, "bwd_read": 16 * 33 * KB, "bwd_red": 16 * 32 * KB},
                  {"fwd_read": 16 * 32 * KB, "bwd_read": 0, "bwd_red": 0}]
    # staged: rank 1 receives K_0, V_0 once (512 rows * 64 * 2 B * 2); rank 0 receives Q_1, dO_1 (128 KB) + LSE, D (4 KB)
    # once and sends one fp32 dQ partial of 512 rows back (128 KB)
    sg = link_bytes([0, 1024], 2, 2, "staged", 1, 1, 64)
    assert sg == [{"fwd_read": 0, "bwd_read": 132 * KB, "bwd_red": 128 * KB}, {"fwd_read": 128 * KB, "bwd_read": 0, "bwd_red": 0}]


def test_gqa_pairs_share_the_stream_and_pair_tiles_at_d128():
    # 8 q-heads on 2 kv-heads: 4 work items per Q tile in the forward (two q-heads share a K/V stream), 8 q-heads in the backward
    a = link_bytes([0, 1024], 2, 2, "stitched", 8, 2, 128)
    assert a[1]["fwd_read"] == 16 * 4 * (2 * 128 * 128 * 2)
    # backward at d = 128 walks 256-key pair-tiles: 2 K/V tiles on rank 0, each streaming the 4 row tiles of rank 1
    assert a[0]["bwd_read"] == 8 * 8 * (2 * 128 * 128 * 2 + 2 * 128 * 4) and a[0]["bwd_red"] == 8 * 8 * 128 * 128 * 4


def test_documents_that_do_not_cross_ranks_move_nothing():
    for design in ("stitched", "staged"):
        for r in link_bytes([0, 512, 1024, 1536, 2048], 4, 4, design, 4, 4, 64):
            assert r == {"fwd_read": 0, "bwd_read": 0, "bwd_red": 0}
        assert link_bytes([0, 2048], 4, 1, design, 4, 4, 64) == [{"fwd_read": 0, "bwd_read": 0, "bwd_red": 0}]
    with pytest.raises(ValueError):
        link_bytes([0, 2048], 4, 3, "staged", 4, 4, 64)


def test_cfg1_and_the_headline_configs(capsys):
    w = make_workload(1)   # 2048 tokens, documents 700 / 1100 / 248, 4 chunks of 512, 4 heads of 64 (MHA)
    st = link_bytes(w.cu_seqlens, 4, 4, "stitched", 4, 4, 64)
    sg = link_bytes(w.cu_seqlens, 4, 4, "staged", 4, 4, 64)
    # forward by hand: rank 1 (rows 512..1023): the 700-token document ends at 700, so its Q tiles 512 and 640 stream the
    # key tiles 0..384 of rank 0 (8 loads); rows from 700 on belong to document 2, which starts on this rank
    # rank 2 (rows 1024..1535, all of document 2 = [700, 1800)): 4 Q tiles x key tiles 640, 768, 896 of rank 1 (12 loads;
    # the tile at 640 holds the document's first key, 700); rank 3 (rows 1536..2047): document 2 up to row 1799 = Q tiles 1536, 1664, 1792
    # x key tiles 640..1408 (7 tiles) = 21 loads; document 3 starts at 1800 on this rank
    per_load = 4 * 2 * 128 * 64 * 2
    assert [r["fwd_read"] // per_load for r in st] == [0, 8, 12, 21]
    # staged: rank 1 gets K/V rows [0, 512) of chunk 0; rank 2 rows [700, 1024) of chunk 1; rank 3 rows [700, 1024) and [1024, 1536)
    per_row = 4 * 64 * 2 * 2
    assert [r["fwd_read"] // per_row for r in sg] == [0, 512, 324, 324 + 512]
    for a, b in zip(st, sg):
        assert all(b[k] <= a[k] for k in a)
    with capsys.disabled():
        print()
        for cfg in (3, 5):
            w = make_workload(cfg)
            q_work, kv_work = chunk_work(w.cu_seqlens, w.n_chunks)
            for world in (2, 4, 8):
                per = w.n_chunks // world
                for design in ("stitched", "staged"):
                    lb = link_bytes(w.cu_seqlens, w.n_chunks, world, design, w.n_q_heads, w.n_kv_heads, w.head_dim)
                    # inbound per rank: what it reads; the fp32 contributions it SENDS arrive at their owners, bounded by the same link
                    worst_f = max(r["fwd_read"] for r in lb)
                    worst_b = max(r["bwd_read"] + r["bwd_red"] for r in lb)
                    f_work = max(sum(q_work[r * per:(r + 1) * per]) for r in range(world)) * 4 * w.head_dim * w.n_q_heads
                    b_work = max(sum(kv_work[r * per:(r + 1) * per]) for r in range(world)) * 10 * w.head_dim * w.n_q_heads
                    print(f"cfg{cfg} {world} ranks {design:8s}: fwd worst rank {worst_f / 1e9:7.2f} GB = {worst_f / 0.9e12 * 1e3:6.2f} ms of link "
                          f"vs {f_work / 1238e12 * 1e3:5.2f} ms of compute; bwd {worst_b / 1e9:7.2f} GB = {worst_b / 0.9e12 * 1e3:6.2f} ms "
                          f"vs {b_work / 1090e12 * 1e3:5.2f} ms")
