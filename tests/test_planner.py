"""Host logic of the library (no GPU): the closed-form planner in libsap_b200.so must match the oracle's
brute-definition planner bit-exactly (pins P11-P13), and reject bad input with the
documented status codes."""
import os

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

import paper_2606_30460_b200 as sap
from oracle import oracle
from paper_2606_30460_b200.workloads import make_workload

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def assert_same_plan(cu, P):
    a = sap.sap_plan(cu, P)
    b = oracle.plan(cu, P)
    assert a.n_items == b.n_items
    assert a.items.tobytes() == b.items.tobytes()
    assert a.chunk_offsets.tobytes() == b.chunk_offsets.tobytes()
    assert a.kv_offsets.tobytes() == b.kv_offsets.tobytes()
    assert a.kv_index.tobytes() == b.kv_index.tobytes()
    assert a.kind_map.tobytes() == b.kind_map.tobytes()
    return a


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_plan_matches_oracle_on_configs(cfg):
    w = make_workload(cfg)
    p = assert_same_plan(w.cu_seqlens, w.n_chunks)
    assert p.useful_pairs == w.pairs


def test_plan_cfg1_matches_survey_appendix_a1():
    # SURVEY Appendix A.1 (derived from BASELINE.json configs[0]): 8 items in ring order
    expect = [(0, 0, 0, 0, 2, 0, 512, 0, 512), (1, 1, 0, 1, 2, 512, 1024, 512, 1024),
              (1, 0, 0, 0, 1, 512, 700, 0, 512), (2, 2, 1, 1, 2, 1024, 1536, 1024, 1536),
              (2, 1, 1, 1, 1, 1024, 1536, 700, 1024), (3, 3, 1, 2, 2, 1536, 2048, 1536, 2048),
              (3, 2, 1, 1, 1, 1536, 1800, 1024, 1536), (3, 1, 1, 1, 1, 1536, 1800, 700, 1024)]
    p = sap.sap_plan([0, 700, 1800, 2048], 4)
    got = [tuple(int(x) for x in (r[0], r[1], r[2], r[3], r[4], r[6], r[7], r[8], r[9])) for r in p.items]
    assert got == expect
    assert [int(r[5]) for r in p.items] == [0, 0, 1, 0, 1, 0, 1, 2]
    assert p.useful_pairs == 881776


def test_single_document_closed_form():
    p = sap.sap_plan([0, 131072], 16)
    kinds = p.items[:, 4]
    assert p.n_items == 136 and int((kinds == 1).sum()) == 120 and int((kinds == 2).sum()) == 16
    assert p.useful_pairs == 8590000128


@settings(max_examples=150, deadline=None)
@given(st.lists(st.integers(0, 40), min_size=1, max_size=12), st.integers(1, 8))
def test_plan_matches_oracle_random(lens, P):
    total = sum(lens)
    if total == 0:
        lens = lens + [P]
        total = P
    pad = (-total) % P
    if pad:
        lens = lens + [pad]
    cu = np.concatenate([[0], np.cumsum(lens)]).tolist()
    assert_same_plan(cu, P)


def test_tile_program_covers_every_visible_pair_once():
    # brute force on a ragged case: replay the fwd tile program's masks on the host and compare with the
    # explicit document & causal mask (each visible pair exactly once, nothing else)
    import ctypes
    from paper_2606_30460_b200 import _lib
    lens = [300, 0, 33, 167]
    cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    N, P = int(cu[-1]), 5
    p = sap.sap_plan(cu.tolist(), P)
    items = p.items
    doc = np.searchsorted(cu, np.arange(N), side="right") - 1
    want = (doc[:, None] == doc[None, :]) & (np.arange(N)[None, :] <= np.arange(N)[:, None])
    count = np.zeros((N, N), dtype=np.int32)
    for it in items:
        qb, qe, kb, ke = (int(x) for x in it[6:10])
        sub = want[qb:qe, kb:ke]
        if it[4] == sap.SAP_MASK_FULL:
            assert sub.all()           # FULL rectangles contain no masked element
        count[qb:qe, kb:ke] += sub.astype(np.int32)
    assert np.array_equal(count, want.astype(np.int32))
    assert p.fwd_tiles >= (want.sum() + 16383) // 16384


@pytest.mark.parametrize("cu,P,status", [([1, 5], 1, 2), ([0, 5, 3], 1, 2), ([0, 0], 1, 2), ([0, 10], 3, 3),
                                         ([0, 10], 0, 1)])
def test_plan_error_codes(cu, P, status):
    with pytest.raises(sap.SapError) as e:
        sap.sap_plan(cu, P)
    assert e.value.status == status
