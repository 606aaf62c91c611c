"""Pins for the oracle's brute-definition planner (pins P11-P14)."""
import os

import numpy as np
import pytest

from oracle import oracle
from paper_2606_30460_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
KIND = {"F": oracle.FULL, "D": oracle.DIAG}


def read_fixture(name):
    docs, chunks, rows, meta = None, None, [], {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            tok = line.split()
            if tok[0] == "docs":
                docs = [int(x) for x in tok[1:]]
            elif tok[0] == "chunks":
                chunks = int(tok[1])
            elif tok[0] in ("n_items", "n_full", "n_skip_causal", "pairs", "n_tokens", "n_docs", "n_chunks"):
                meta[tok[0]] = int(tok[1])
            elif tok[0] == "sha256":
                meta["sha256"] = tok[1]
            else:
                rows.append(tok)
    return docs, chunks, rows, meta


def cu_of(docs):
    return np.concatenate([[0], np.cumsum(docs)]).astype(np.int32)


def allowed_pairs_of_item(it, cu):
    """Number of (row, key) pairs an item covers under the document-and-causal mask."""
    qb, qe, kb, ke = (int(x) for x in it[6:10])
    tot = 0
    for e in range(len(cu) - 1):
        r0, r1 = max(cu[e], qb), min(cu[e + 1], qe)
        c0, c1 = max(cu[e], kb), min(cu[e + 1], ke)
        if r0 >= r1 or c0 >= c1:
            continue
        for t in range(r0, r1):
            hi = min(t, c1 - 1)
            if hi >= c0:
                tot += hi - c0 + 1
    return tot


def test_p13_worked_plan_a1_cfg1():
    docs, P, rows, _ = read_fixture("plan_a1_cfg1.txt")
    cu = cu_of(docs)
    pl = oracle.plan(cu, P)
    assert pl.n_items == len(rows) == 8
    total = 0
    for it, row in zip(pl.items, rows):
        i, j, dlo, dhi = (int(x) for x in row[:4])
        qb, qe, kb, ke, pairs = (int(x) for x in row[5:10])
        assert list(it) == [i, j, dlo, dhi, KIND[row[4]], i - j, qb, qe, kb, ke]
        assert allowed_pairs_of_item(it, cu) == pairs
        total += pairs
    assert total == 881776                                        # P14
    assert pl.kind_map[2, 0] == oracle.SKIP and pl.kind_map[3, 0] == oracle.SKIP
    assert list(pl.chunk_offsets) == [0, 1, 3, 5, 8]
    assert list(pl.kv_offsets) == [0, 2, 5, 7, 8]
    assert list(pl.kv_index) == [0, 2, 1, 4, 7, 3, 6, 5]


@pytest.mark.parametrize("name", ["plan_a2.txt", "plan_a3.txt"])
def test_p13_worked_plans_a2_a3(name):
    docs, P, rows, meta = read_fixture(name)
    cu = cu_of(docs)
    pl = oracle.plan(cu, P)
    assert pl.n_items == meta["n_items"]
    assert int((pl.items[:, 4] == oracle.FULL).sum()) == meta["n_full"]
    assert int((pl.items[:, 4] == oracle.DIAG).sum()) == P
    n_skip = sum(1 for i in range(P) for j in range(i + 1) if pl.kind_map[i, j] == oracle.SKIP)
    assert n_skip == meta["n_skip_causal"]
    assert sum(L * (L + 1) // 2 for L in docs) == meta["pairs"]
    by = {(int(it[0]), int(it[1])): it for it in pl.items}
    for row in rows:
        if row[0] == "F":
            i, j, dlo, dhi, qb, qe, kb, ke = (int(x) for x in row[1:])
            assert list(by[(i, j)]) == [i, j, dlo, dhi, oracle.FULL, i - j, qb, qe, kb, ke]
        elif row[0] == "D":
            i, dlo, dhi = (int(x) for x in row[1:])
            it = by[(i, i)]
            assert (int(it[2]), int(it[3]), int(it[4])) == (dlo, dhi, oracle.DIAG)
        elif row[0] == "M":
            i = int(row[1])
            sel = pl.items[pl.chunk_offsets[i]:pl.chunk_offsets[i + 1]]
            assert [int(x[1]) for x in sel if x[4] == oracle.FULL] == [int(x) for x in row[2:]]
        elif row[0] == "R":
            i, qb, qe = (int(x) for x in row[1:])
            sel = pl.items[pl.chunk_offsets[i]:pl.chunk_offsets[i + 1]]
            for x in sel:
                if x[4] == oracle.FULL:
                    assert (int(x[6]), int(x[7])) == (qb, qe)


def explicit_mask(cu, N):
    idx = np.arange(N)
    doc = np.searchsorted(cu, idx, side="right") - 1
    return (doc[:, None] == doc[None, :]) & (idx[None, :] <= idx[:, None])


@pytest.mark.parametrize("docs,P", [([5, 9, 1, 12, 3], 5), ([30], 6), ([4, 4, 4, 4], 4), ([3, 0, 7, 0, 0, 6], 4),
                                    ([1] * 24, 3), ([17, 2, 29], 2), ([7, 20, 3, 18], 12), ([11, 13], 1)])
def test_p11_plan_covers_the_mask_exactly_once(docs, P):
    cu = cu_of(docs)
    N = int(cu[-1])
    mask = explicit_mask(cu, N)
    pl = oracle.plan(cu, P)
    cover = np.zeros((N, N), dtype=np.int32)
    for it in pl.items:
        i, j, dlo, dhi, kind, step, qb, qe, kb, ke = (int(x) for x in it)
        assert step == i - j and kind == (oracle.DIAG if i == j else oracle.FULL)
        sub = mask[qb:qe, kb:ke]
        cover[qb:qe, kb:ke] += sub
        if kind == oracle.FULL:
            assert sub.all(), "a FULL rectangle must contain no masked element"
        # everything of the chunk pair outside the item's rectangle is masked
        n = N // P
        blk = mask[i * n:(i + 1) * n, j * n:(j + 1) * n].copy()
        blk[qb - i * n:qe - i * n, kb - j * n:ke - j * n] = False
        assert not blk.any()
        # doc range: exactly the documents with an allowed pair in the rectangle
        rows_docs = set(np.searchsorted(cu, np.nonzero(sub.any(axis=1))[0] + qb, side="right") - 1)
        assert min(rows_docs) == dlo and max(rows_docs) == dhi
    np.testing.assert_array_equal(cover, mask.astype(np.int32))
    # SKIP pairs: no allowed element at all; kind map agrees with the list
    n = N // P
    listed = {(int(it[0]), int(it[1])) for it in pl.items}
    for i in range(P):
        for j in range(P):
            blk = mask[i * n:(i + 1) * n, j * n:(j + 1) * n]
            if (i, j) in listed:
                assert pl.kind_map[i, j] != oracle.SKIP
            else:
                assert pl.kind_map[i, j] == oracle.SKIP and not blk.any()


def test_p12_closed_forms():
    # single document: P(P+1)/2 items, P DIAG, rest FULL, none skipped (cfg4: 120 FULL + 16 DIAG)
    pl = oracle.plan(np.array([0, 131072], dtype=np.int32), 16)
    assert pl.n_items == 136 and int((pl.items[:, 4] == oracle.FULL).sum()) == 120
    assert int((pl.items[:, 4] == oracle.DIAG).sum()) == 16
    assert all(pl.kind_map[i, j] != oracle.SKIP for i in range(16) for j in range(i + 1))
    assert all(pl.kind_map[i, j] == oracle.SKIP for i in range(16) for j in range(i + 1, 16))
    # P = 1: one DIAG item spanning everything
    pl = oracle.plan(cu_of([5, 6, 7]), 1)
    assert pl.items.tolist() == [[0, 0, 0, 2, oracle.DIAG, 0, 0, 18, 0, 18]]
    # a document starting exactly at i*n: chunk i has only its DIAG item
    pl = oracle.plan(cu_of([16, 16, 32]), 4)
    for i in (1, 2):
        sel = pl.items[pl.chunk_offsets[i]:pl.chunk_offsets[i + 1]]
        assert len(sel) == 1 and sel[0][4] == oracle.DIAG
    sel = pl.items[pl.chunk_offsets[3]:pl.chunk_offsets[4]]
    assert [(int(x[1]), int(x[4])) for x in sel] == [(3, oracle.DIAG), (2, oracle.FULL)]


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_p12_p14_pair_totals_and_fixtures(cfg):
    docs, _, _, meta = read_fixture(f"cu_seqlens_cfg{cfg}.txt")
    w = W.make_workload(cfg)
    assert list(w.doc_lens) == docs and w.sha256() == meta["sha256"]
    assert w.pairs == meta["pairs"] == sum(L * (L + 1) // 2 for L in docs)
    if cfg == 1:
        assert w.pairs == 881776
    if cfg == 4:
        assert w.pairs == 8590000128
    pl = oracle.plan(w.cu_seqlens, w.n_chunks)
    # sum over items of allowed pairs == sum over docs L(L+1)/2, via the closed form of each item:
    # FULL rectangles are unmasked (P11), DIAG blocks are block-diagonal causal.
    cu = np.array(w.cu_seqlens, dtype=np.int64)
    tot = 0
    for it in pl.items:
        i, j, dlo, dhi, kind, step, qb, qe, kb, ke = (int(x) for x in it)
        if kind == oracle.FULL:
            tot += (qe - qb) * (ke - kb)
        else:
            for e in range(dlo, dhi + 1):
                a, b = max(cu[e], qb), min(cu[e + 1], qe)
                L = b - a
                if L > 0:
                    tot += L * (L + 1) // 2
    assert tot == w.pairs


def test_plan_rejects_bad_input():
    with pytest.raises(ValueError):
        oracle.plan([0, 10], 3)                       # N % P != 0
    with pytest.raises(ValueError):
        oracle.plan([1, 10], 1)                       # cu[0] != 0
    with pytest.raises(ValueError):
        oracle.plan([0, 10, 5], 1)                    # decreasing
    with pytest.raises(ValueError):
        oracle.plan([0, 10], 0)
