"""The compiled tile programs (TileDesc / SegDesc: what the kernels actually walk) replayed on the host: every visible
(row, key) pair of the items a program covers is computed by exactly one (tile, segment), nothing else is - for the
full programs (forward, backward with 128- and 256-key tiles) and for every restricted variant (item ranges, q-chunk
and kv-chunk ranges).  Seeded random packings with chunk lengths that are not tile multiples and zero-length documents."""
import numpy as np
import pytest

import paper_2606_30460_b200 as sap

KV_KINDS = {1, 2, 6, 7, 8, 9}


def visible_matrix(cu, items, item_ids):
    N = cu[-1]
    doc = np.searchsorted(np.asarray(cu), np.arange(N), side="right") - 1
    t, s = np.arange(N)[:, None], np.arange(N)[None, :]
    same = (doc[:, None] == doc[None, :]) & (s <= t)
    want = np.zeros((N, N), dtype=np.int32)
    for x in item_ids:
        qb, qe, kb, ke = (int(v) for v in items[x, 6:10])
        want[qb:qe, kb:ke] += same[qb:qe, kb:ke]
    return want, same


def replay(plan, cu, kind, a=0, b=0):
    tiles, segs = plan.tile_program(kind, a, b)
    N = cu[-1]
    got = np.zeros((N, N), dtype=np.int32)
    _, same = visible_matrix(cu, plan.items, [])
    for row0, rows, sb, se in tiles.tolist():
        st = np.arange(row0, row0 + rows)                      # stationary indices of the tile
        for t_begin, t_end, q_lo, q_hi, kv_lo, kv_hi, item, _ in segs[sb:se].tolist():
            mv = np.arange(t_begin, min(t_end, N))              # streamed indices
            if kind in KV_KINDS:                                # K/V-stationary: tile = keys, streamed = rows
                tt, ss = mv[(mv >= q_lo) & (mv < q_hi)], st[(st >= kv_lo) & (st < kv_hi)]
            else:
                tt, ss = st[(st >= q_lo) & (st < q_hi)], mv[(mv >= kv_lo) & (mv < kv_hi)]
            if len(tt) and len(ss):
                got[np.ix_(tt, ss)] += same[np.ix_(tt, ss)]
    return got, tiles


def random_layout(rng):
    P = int(rng.integers(1, 9))
    n = int(rng.choice([96, 128, 200, 256, 384, 512]))
    N = P * n
    k = int(rng.integers(1, 8))
    cuts = np.sort(rng.integers(0, N + 1, size=k - 1)) if k > 1 else np.array([], dtype=np.int64)
    cu = [0] + [int(c) for c in cuts] + [N]                    # repeated entries = zero-length documents
    return cu, P


@pytest.mark.parametrize("seed", range(24))
def test_every_visible_pair_is_covered_exactly_once(seed):
    rng = np.random.default_rng(1000 + seed)
    cu, P = random_layout(rng)
    plan = sap.sap_plan(cu, P)
    items, n_items = plan.items, plan.n_items
    all_items = list(range(n_items))
    want_all, _ = visible_matrix(cu, items, all_items)
    assert want_all.max() <= 1                                   # items are disjoint (oracle pin P11 on the library's plan)
    for kind in (0, 1, 2, 10):                                   # the programs sap_attn_fwd / sap_attn_bwd walk (10: 256-row Q tiles)
        got, _ = replay(plan, cu, kind)
        assert np.array_equal(got, want_all), (kind, cu, P)
    a = int(rng.integers(0, n_items)); b = int(rng.integers(a, n_items + 1))
    want_ab, _ = visible_matrix(cu, items, range(a, b))
    for kind in (3, 4, 8, 9):                                    # item ranges: partial forward, forward / backward `computing`
        got, tiles = replay(plan, cu, kind, a, b)
        assert np.array_equal(got, want_ab), (kind, a, b, cu, P)
        if kind != 3 and a == b:
            assert len(tiles) == 0
    ca = int(rng.integers(0, P)); cb = int(rng.integers(ca, P + 1))
    co = plan.chunk_offsets
    want_q, _ = visible_matrix(cu, items, range(int(co[ca]), int(co[cb])))
    got, tiles = replay(plan, cu, 5, ca, cb)                      # a rank's forward: its q-chunks
    assert np.array_equal(got, want_q)
    n = cu[-1] // P
    assert all(ca * n <= r0 and r0 + rows <= cb * n for r0, rows, _, _ in tiles.tolist())    # writes only its own rows
    kv_items = [x for x in all_items if ca <= int(items[x, 1]) < cb]
    want_kv, _ = visible_matrix(cu, items, kv_items)
    for kind in (6, 7):                                          # a rank's backward: its kv-chunks
        got, tiles = replay(plan, cu, kind, ca, cb)
        assert np.array_equal(got, want_kv), (kind, ca, cb, cu, P)
        assert all(ca * n <= r0 and r0 + rows <= cb * n for r0, rows, _, _ in tiles.tolist())


def test_pair_tiles_are_256_keys_from_the_range_start():
    plan = sap.sap_plan([0, 700, 1800, 2048], 4)
    tiles, _ = plan.tile_program(2)
    assert sorted(t[0] for t in tiles.tolist()) == list(range(0, 2048, 256)) and all(t[1] == 256 for t in tiles.tolist())
    tiles, _ = plan.tile_program(7, 1, 3)                         # kv-chunks 1..2: rows 512..1535
    assert sorted(t[0] for t in tiles.tolist()) == [512, 768, 1024, 1280]


def _work(tiles, segs, tile_rows=128):
    return [sum((te - tb + 127) // 128 for tb, te, *_ in segs[sb:se].tolist()) for _, _, sb, se in tiles.tolist()]


@pytest.mark.parametrize("kind", [1, 2])
def test_kv_tiles_are_launched_document_by_document(kind):
    """Launch order of the KV-stationary programs: the tiles whose last key lies in one document
    are adjacent, documents in order of their longest tile, and inside a document longest tile first - so the rows the
    concurrently running tiles add into (that document's part of the dQ accumulator) stay in L2."""
    cu = [0, 300, 300, 2900, 3000, 7000, 7100, 8192]
    plan = sap.sap_plan(cu, 8)
    tiles, segs = plan.tile_program(kind)
    work = _work(tiles, segs)
    doc = [int(np.searchsorted(np.asarray(cu), r0 + rows - 1, side="right") - 1) for r0, rows, _, _ in tiles.tolist()]
    seen, prev = [], None
    for d in doc:                                                # contiguous groups
        if d != prev:
            assert d not in seen, (doc, "tiles of one document are not adjacent")
            seen.append(d); prev = d
    best = {d: max(w for w, dd in zip(work, doc) if dd == d) for d in seen}
    assert [best[d] for d in seen] == sorted((best[d] for d in seen), reverse=True)      # documents: longest tile first
    for d in seen:
        w = [x for x, dd in zip(work, doc) if dd == d]
        assert w == sorted(w, reverse=True)                      # inside a document: longest first


def test_q_tiles_are_longest_first_below_the_grouping_threshold():
    """The Q-stationary program of a sequence below 192K tokens is plain longest-first (sap_plan.cpp:
    kGroupQTilesFromTokens); from there on its tiles are grouped by the document of their first row."""
    plan = sap.sap_plan([0, 300, 2900, 3000, 7000, 8192], 8)
    tiles, segs = plan.tile_program(0)
    work = _work(tiles, segs)
    assert work == sorted(work, reverse=True)
    big = [0, 100_000, 150_000, 196_608]                        # 192K tokens: grouped
    plan = sap.sap_plan(big, 8)
    tiles, segs = plan.tile_program(0)
    doc = [int(np.searchsorted(np.asarray(big), r0, side="right") - 1) for r0, _, _, _ in tiles.tolist()]
    changes = sum(1 for a, b in zip(doc, doc[1:]) if a != b)
    assert changes == 2 and doc[0] == 0                          # three groups, the 100K-token document first
