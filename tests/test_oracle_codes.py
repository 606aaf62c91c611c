"""Pins of the oracle's instruction-list checker (oracle.check_codes) with hand-made lists: one legal list per transport
pattern of Table 1 written out by hand from the paper's description of the execute side (:100-102,
:120-124), and for each rule a mutation that must be caught.  The checker shares nothing with sap_plan_codegen."""
import numpy as np

from oracle import oracle
from oracle.oracle import OP_COMPUTING as C, OP_COPY as CP, OP_RECV as R, OP_SEND as S, T_DKV, T_DO, T_DQ, T_KV, T_O, T_Q

CU, P = [0, 256], 2                      # one document over two chunks: items 0 = (0,0) DIAG, 1 = (1,1) DIAG, 2 = (1,0) FULL


def arr(codes):
    return [np.array(c, dtype=np.int32).reshape(-1, 5) for c in codes]


def test_plan_of_the_hand_made_case():
    pl = oracle.plan(CU, P)
    assert [(int(r[0]), int(r[1])) for r in pl.items] == [(0, 0), (1, 1), (1, 0)]


RING_SLOTS = [(0, 0), (1, 0), (1, 1)]    # item (1,0) on rank 1 (the rank of its Q) at stage 1
RING_FWD = [
    [(0, S, T_KV, 1, 2), (0, C, -1, -1, 0)],                                            # rank 0: K/V_0 leaves while block (0,0) runs
    [(0, R, T_KV, 0, 2), (0, C, -1, -1, 1), (0, CP, T_KV, 0, 2), (1, C, -1, -1, 2)],    # rank 1: receive, compute (1,1), copy, compute (1,0)
]
HELP_SLOTS = [(0, 0), (1, 0), (0, 1)]    # item (1,0) on rank 0 (the rank of its K/V): Q_1 travels, the partial comes back
HELP_FWD = [
    [(0, R, T_Q, 1, 2), (0, C, -1, -1, 0), (0, CP, T_Q, 1, 2), (1, C, -1, -1, 2), (2, S, T_O, 1, 2)],
    [(0, S, T_Q, 0, 2), (0, C, -1, -1, 1), (2, R, T_O, 0, 2), (2, CP, T_O, 0, 2)],
]


def test_hand_made_legal_lists_pass():
    assert oracle.check_codes(CU, P, RING_SLOTS, arr(RING_FWD)) == []
    assert oracle.check_codes(CU, P, HELP_SLOTS, arr(HELP_FWD)) == []
    # later stages than strictly necessary are still legal (the checker does not prescribe stage offsets)
    late = [HELP_FWD[0][:-1] + [(5, S, T_O, 1, 2)], HELP_FWD[1][:2] + [(5, R, T_O, 0, 2), (7, CP, T_O, 0, 2)]]
    assert oracle.check_codes(CU, P, HELP_SLOTS, arr(late)) == []


def first_rule(bad):
    assert bad, "the mutation was not caught"
    return bad[0][:2]


def test_mutations_are_caught_rule_by_rule():
    # R3: the operand is copied in the stage it is used in (not before)
    m = [RING_FWD[0], [(0, R, T_KV, 0, 2), (0, C, -1, -1, 1), (1, C, -1, -1, 2), (1, CP, T_KV, 0, 2)]]
    assert any(b.startswith("R3") for b in oracle.check_codes(CU, P, RING_SLOTS, arr(m)))
    # R4: a SEND without its RECV
    m = [RING_FWD[0], [c for c in RING_FWD[1] if c[1] not in (R, CP)]]
    assert any(b.startswith("R4") for b in oracle.check_codes(CU, P, RING_SLOTS, arr(m)))
    # R4: RECV at another stage than the SEND
    m = [RING_FWD[0], [(1, R, T_KV, 0, 2) if c[1] == R else c for c in RING_FWD[1]]]
    assert oracle.check_codes(CU, P, RING_SLOTS, arr(m)) != []
    # R2: an item computed on the wrong rank / twice / not at all
    m = [RING_FWD[0] + [(1, C, -1, -1, 2)], RING_FWD[1]]
    assert any(b.startswith("R2") for b in oracle.check_codes(CU, P, RING_SLOTS, arr(m)))
    m = [RING_FWD[0], RING_FWD[1][:-1]]
    assert any(b.startswith("R2") for b in oracle.check_codes(CU, P, RING_SLOTS, arr(m)))
    # R5: the helper's partial is never returned / returned before it exists
    m = [HELP_FWD[0][:-1], HELP_FWD[1][:2]]
    assert any(b.startswith("R5") for b in oracle.check_codes(CU, P, HELP_SLOTS, arr(m)))
    m = [HELP_FWD[0][:-1] + [(1, S, T_O, 1, 2)], HELP_FWD[1][:2] + [(1, R, T_O, 0, 2), (1, CP, T_O, 0, 2)]]
    m[0] = sorted(m[0], key=lambda c: (c[0], {S: 0, R: 0, C: 1, CP: 2}[c[1]]))
    assert any(b.startswith("R5") for b in oracle.check_codes(CU, P, HELP_SLOTS, arr(m)))
    # R1: COPY before COMPUTING inside a stage
    m = [RING_FWD[0], [(0, R, T_KV, 0, 2), (0, CP, T_KV, 0, 2), (0, C, -1, -1, 1), (1, C, -1, -1, 2)]]
    assert any(b.startswith("R1") for b in oracle.check_codes(CU, P, RING_SLOTS, arr(m)))
    # R3/R5: a transfer nobody needs (K/V sent although the helper form is scheduled)
    m = [[(0, S, T_KV, 1, 2)] + HELP_FWD[0], [(0, R, T_KV, 0, 2)] + HELP_FWD[1][:2] + [(0, CP, T_KV, 0, 2)] + HELP_FWD[1][2:]]
    m[1] = sorted(m[1], key=lambda c: (c[0], {S: 0, R: 0, C: 1, CP: 2}[c[1]]))
    assert any("nobody needs" in b for b in oracle.check_codes(CU, P, HELP_SLOTS, arr(m)))


def test_backward_lists():
    ring = [
        [(0, S, T_KV, 1, 2), (0, C, -1, -1, 0), (2, R, T_DKV, 1, 2), (2, CP, T_DKV, 1, 2)],
        [(0, R, T_KV, 0, 2), (0, C, -1, -1, 1), (0, CP, T_KV, 0, 2), (1, C, -1, -1, 2), (2, S, T_DKV, 0, 2)],
    ]
    assert oracle.check_codes(CU, P, RING_SLOTS, arr(ring), backward=True) == []
    helper = [
        [(0, R, T_Q, 1, 2), (0, R, T_DO, 1, 2), (0, C, -1, -1, 0), (0, CP, T_Q, 1, 2), (0, CP, T_DO, 1, 2), (1, C, -1, -1, 2), (2, S, T_DQ, 1, 2)],
        [(0, S, T_Q, 0, 2), (0, S, T_DO, 0, 2), (0, C, -1, -1, 1), (2, R, T_DQ, 0, 2), (2, CP, T_DQ, 0, 2)],
    ]
    assert oracle.check_codes(CU, P, HELP_SLOTS, arr(helper), backward=True) == []
    no_do = [[c for c in helper[0] if c[2] != T_DO], [c for c in helper[1] if c[2] != T_DO]]
    assert any(b.startswith("R3") for b in oracle.check_codes(CU, P, HELP_SLOTS, arr(no_do), backward=True))   # dO (with LSE, D) must travel with Q
    no_dkv = [ring[0][:2], ring[1][:-1]]
    assert any(b.startswith("R5") for b in oracle.check_codes(CU, P, RING_SLOTS, arr(no_dkv), backward=True))
