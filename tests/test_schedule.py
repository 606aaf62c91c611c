"""Compile Steps 2-3: sap_plan_schedule against the oracle's step-by-step
version (bit-exact) and against what any valid schedule must satisfy, plus the closed forms of the balanced policy."""
import numpy as np
import pytest

import paper_2606_30460_b200 as sap
from oracle import oracle
from paper_2606_30460_b200.workloads import make_workload

LAYOUTS = [([2048], 4), ([2048], 7 * 0 + 8), ([700, 1100, 248], 4), ([100, 1948], 8), ([1000, 24, 1024], 16),
           ([64] * 32, 8), ([3000, 1000, 96], 16), ([1, 4095], 4)]


def cu_of(docs):
    return np.concatenate([[0], np.cumsum(docs)]).astype(np.int64).tolist()


def check_valid(plan, slots, n_stages, balanced):
    items = plan.items
    assert slots.shape == (plan.n_items, 2)
    seen = set()
    for x in range(plan.n_items):
        i, j, kind = int(items[x, 0]), int(items[x, 1]), int(items[x, 4])
        r, st = int(slots[x, 0]), int(slots[x, 1])
        assert r in ((i, j) if balanced else (i,)), "an item runs where its Q or its K/V lives"
        if kind == sap.SAP_MASK_DIAG:
            assert r == i
        assert 0 <= st < n_stages
        assert (r, st) not in seen, "one item per rank and stage"
        seen.add((r, st))
    assert n_stages == (int(slots[:, 1].max()) + 1 if plan.n_items else 0)


@pytest.mark.parametrize("docs,P", LAYOUTS)
@pytest.mark.parametrize("policy", [0, 1])
def test_schedule_matches_oracle_and_is_valid(docs, P, policy):
    cu = cu_of(docs)
    plan = sap.sap_plan(cu, P)
    slots, n_stages = plan.schedule(policy)
    ref_slots, ref_n = oracle.schedule(cu, P, policy)
    assert slots.tobytes() == ref_slots.tobytes() and n_stages == ref_n
    check_valid(plan, slots, n_stages, balanced=(policy == 1))
    # any schedule needs at least ceil(items / ranks) stages and at least the busiest diagonal + ... lower bound
    assert n_stages >= -(-plan.n_items // P)


@pytest.mark.parametrize("P", [1, 2, 3, 4, 7, 8, 16, 64])
def test_single_document_closed_form(P):
    # one causal region over all ranks: the ring needs P stages, the balanced schedule floor(P/2) + 1, loads within 1
    plan = sap.sap_plan([0, 64 * P], P)
    ring, n_ring = plan.schedule(sap.SAP_SCHED_RING)
    bal, n_bal = plan.schedule(sap.SAP_SCHED_BALANCED)
    assert n_ring == P and n_bal == P // 2 + 1
    loads = np.bincount(bal[:, 0], minlength=P)
    assert loads.max() - loads.min() <= 1 and loads.sum() == P * (P + 1) // 2
    assert np.bincount(ring[:, 0], minlength=P).max() == P


@pytest.mark.parametrize("cfg", [2, 3, 4, 5])
def test_balanced_never_worse_than_ring_on_configs(cfg):
    w = make_workload(cfg)
    plan = sap.sap_plan(w.cu_seqlens, w.n_chunks)
    ring, n_ring = plan.schedule(0)
    bal, n_bal = plan.schedule(1)
    ref, ref_n = oracle.schedule(w.cu_seqlens, w.n_chunks, 1)
    assert bal.tobytes() == ref.tobytes() and n_bal == ref_n
    check_valid(plan, bal, n_bal, True)
    assert n_bal <= n_ring
    assert n_bal == np.bincount(bal[:, 0], minlength=w.n_chunks).max()      # no idle stage on the busiest rank
    assert np.bincount(bal[:, 0], minlength=w.n_chunks).max() <= np.bincount(ring[:, 0], minlength=w.n_chunks).max()


def test_schedule_rejects_bad_arguments():
    plan = sap.sap_plan([0, 256], 2)
    with pytest.raises(sap.SapError):
        plan.schedule(7)
