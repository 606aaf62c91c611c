"""Pins for the fp64 oracle's float functions (pins P1-P10).

None of these re-type the oracle's row loop: they compare it with the full-matrix
textbook form, with closed forms, with invariants the paper's claims imply
(PAPER.md:45 no cross-contamination, :29 exact attention, :59 online merge) and with
finite differences.
"""
import numpy as np
import pytest

from oracle import oracle

RNG = np.random.default_rng(1234)


def bf16_exact(a):
    """Round to values representable in bf16 (8 significant bits), kept as float32."""
    a = np.asarray(a, dtype=np.float32)
    u = a.view(np.uint32).astype(np.uint64)
    u = ((u + 0x7FFF + ((u >> 16) & 1)) >> 16) << 16
    return u.astype(np.uint32).view(np.float32).reshape(a.shape)


def make(doc_lens, Hq, Hkv, d, seed=0):
    rng = np.random.default_rng(seed)
    N = int(sum(doc_lens))
    cu = np.concatenate([[0], np.cumsum(doc_lens)]).astype(np.int32)
    q = bf16_exact(rng.standard_normal((N, Hq, d)))
    k = bf16_exact(rng.standard_normal((N, Hkv, d)))
    v = bf16_exact(rng.standard_normal((N, Hkv, d)))
    do = bf16_exact(rng.standard_normal((N, Hq, d)))
    return cu, q, k, v, do


def brute(q, k, v, cu, scale, dout=None):
    """Full N x N attention with an EXPLICIT document-and-causal mask, matrix form, fp64."""
    q = q.astype(np.float64); k = k.astype(np.float64); v = v.astype(np.float64)
    N, Hq, d = q.shape
    Hkv = k.shape[1]
    g = Hq // Hkv
    idx = np.arange(N)
    doc = np.searchsorted(cu, idx, side="right") - 1
    mask = (doc[:, None] == doc[None, :]) & (idx[None, :] <= idx[:, None])
    O = np.zeros((N, Hq, d)); LSE = np.zeros((N, Hq))
    dQ = np.zeros((N, Hq, d)); dK = np.zeros((N, Hkv, d)); dV = np.zeros((N, Hkv, d))
    for h in range(Hq):
        hk = h // g
        S = scale * q[:, h] @ k[:, hk].T
        S = np.where(mask, S, -np.inf)
        m = S.max(axis=1, keepdims=True)
        E = np.exp(S - m)
        l = E.sum(axis=1, keepdims=True)
        P = E / l
        O[:, h] = P @ v[:, hk]
        LSE[:, h] = (m + np.log(l))[:, 0]
        if dout is not None:
            dO = dout[:, h].astype(np.float64)
            dP = dO @ v[:, hk].T
            D = (dO * O[:, h]).sum(axis=1, keepdims=True)
            dS = P * (dP - D)
            dQ[:, h] = scale * dS @ k[:, hk]
            dK[:, hk] += scale * dS.T @ q[:, h]
            dV[:, hk] += P.T @ dO
    return O, LSE, dQ, dK, dV


LAYOUTS = [
    ([17], 2, 2, 8),
    ([5, 9, 1, 12], 4, 2, 8),
    ([1, 1, 1, 30, 2], 4, 1, 16),
    ([20, 20, 24], 2, 2, 4),
    ([3, 0, 7, 0, 0, 6], 2, 1, 8),        # zero-length documents (reading A-9)
]


@pytest.mark.parametrize("docs,Hq,Hkv,d", LAYOUTS)
def test_p1_brute_force_full_matrix(docs, Hq, Hkv, d):
    cu, q, k, v, do = make(docs, Hq, Hkv, d, seed=len(docs))
    scale = 1.0 / np.sqrt(d)
    O, LSE, dQ, dK, dV = brute(q, k, v, cu, scale, do)
    o, lse = oracle.attn_fwd(q, k, v, cu, scale)
    np.testing.assert_allclose(o, O, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(lse, LSE, rtol=1e-12, atol=1e-13)
    dq = oracle.attn_bwd_dq(q, k, v, do, cu, scale)
    dk, dv = oracle.attn_bwd_dkv(q, k, v, do, cu, scale)
    np.testing.assert_allclose(dq, dQ, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(dk, dK, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(dv, dV, rtol=1e-11, atol=1e-12)


def test_p1_row_and_column_subsets_match_full():
    cu, q, k, v, do = make([9, 14, 6], 4, 2, 8, seed=5)
    scale = 0.3
    rows = np.array([0, 8, 9, 22, 23, 28], dtype=np.int64)
    o, lse = oracle.attn_fwd(q, k, v, cu, scale)
    o_s, lse_s = oracle.attn_fwd(q, k, v, cu, scale, rows)
    np.testing.assert_array_equal(o_s, o[rows]); np.testing.assert_array_equal(lse_s, lse[rows])
    dq = oracle.attn_bwd_dq(q, k, v, do, cu, scale)
    np.testing.assert_array_equal(oracle.attn_bwd_dq(q, k, v, do, cu, scale, rows), dq[rows])
    dk, dv = oracle.attn_bwd_dkv(q, k, v, do, cu, scale)
    dk_s, dv_s = oracle.attn_bwd_dkv(q, k, v, do, cu, scale, rows)
    np.testing.assert_allclose(dk_s, dk[rows], rtol=1e-14); np.testing.assert_allclose(dv_s, dv[rows], rtol=1e-14)


def test_p2_packed_equals_each_document_alone():
    docs = [11, 1, 25, 8]
    cu, q, k, v, do = make(docs, 4, 2, 8, seed=7)
    scale = 1.0 / np.sqrt(8)
    o, lse = oracle.attn_fwd(q, k, v, cu, scale)
    dq = oracle.attn_bwd_dq(q, k, v, do, cu, scale)
    dk, dv = oracle.attn_bwd_dkv(q, k, v, do, cu, scale)
    for e, L in enumerate(docs):
        a, b = cu[e], cu[e + 1]
        one = np.array([0, L], dtype=np.int32)
        o1, l1 = oracle.attn_fwd(q[a:b], k[a:b], v[a:b], one, scale)
        np.testing.assert_allclose(o[a:b], o1, rtol=1e-14, atol=0)
        np.testing.assert_allclose(lse[a:b], l1, rtol=1e-14, atol=0)
        np.testing.assert_allclose(dq[a:b], oracle.attn_bwd_dq(q[a:b], k[a:b], v[a:b], do[a:b], one, scale), rtol=1e-13)
        dk1, dv1 = oracle.attn_bwd_dkv(q[a:b], k[a:b], v[a:b], do[a:b], one, scale)
        np.testing.assert_allclose(dk[a:b], dk1, rtol=1e-13); np.testing.assert_allclose(dv[a:b], dv1, rtol=1e-13)


@pytest.mark.parametrize("P", [1, 2, 3, 4, 6, 12])
def test_p3_any_chunking_plus_merge_equals_unchunked(P):
    """per-rank Q shards against incoming K/V shards, merged online -> exact (:29)."""
    docs = [7, 20, 3, 18]                       # N = 48, divisible by every P above
    cu, q, k, v, _ = make(docs, 4, 2, 8, seed=P)
    scale = 0.35
    o_ref, lse_ref = oracle.attn_fwd(q, k, v, cu, scale)
    pl = oracle.plan(cu, P)
    N = q.shape[0]
    o_acc = np.zeros_like(o_ref)
    lse_acc = np.full_like(lse_ref, -np.inf)
    for it in pl.items:
        qb, qe, kb, ke = (int(x) for x in it[6:10])
        o_p, lse_p = oracle.attn_partial(q, k, v, cu, scale, qb, qe, kb, ke)
        o_acc[qb:qe], lse_acc[qb:qe] = oracle.lse_merge(o_acc[qb:qe], lse_acc[qb:qe], o_p, lse_p)
    np.testing.assert_allclose(o_acc, o_ref, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(lse_acc, lse_ref, rtol=1e-13, atol=1e-14)


def test_p4_softmax_rows_sum_to_one_constant_v():
    cu, q, k, v, _ = make([13, 29, 6], 4, 4, 8, seed=3)
    v[:] = 0.75
    o, _ = oracle.attn_fwd(q, k, v, cu, 0.5)
    np.testing.assert_allclose(o, 0.75, rtol=1e-14)


def test_p5_finite_differences_of_backward():
    """Central differences with Richardson extrapolation; perturbations 2^-8, 2^-9 are exact in fp32."""
    docs = [4, 6, 1]
    cu, q, k, v, do = make(docs, 2, 1, 4, seed=11)
    scale = 0.5

    def loss(q_, k_, v_):
        o, _ = oracle.attn_fwd(q_, k_, v_, cu, scale)
        return float((o * do.astype(np.float64)).sum())

    dq = oracle.attn_bwd_dq(q, k, v, do, cu, scale)
    dk, dv = oracle.attn_bwd_dkv(q, k, v, do, cu, scale)
    for name, arr, grad in (("q", q, dq), ("k", k, dk), ("v", v, dv)):
        it = np.nditer(arr, flags=["multi_index"])
        for _ in it:
            ix = it.multi_index
            est = []
            for h in (2.0 ** -8, 2.0 ** -9):
                vals = []
                for sgn in (+1, -1):
                    a = arr.copy(); a[ix] += np.float32(sgn * h)
                    args = {"q": q, "k": k, "v": v}; args[name] = a
                    vals.append(loss(args["q"], args["k"], args["v"]))
                est.append((vals[0] - vals[1]) / (2 * h))
            fd = (4 * est[1] - est[0]) / 3.0
            assert abs(fd - grad[ix]) <= 1e-8 + 1e-7 * abs(grad[ix]), (name, ix, fd, grad[ix])


def test_p6_q_zero_closed_form():
    docs = [5, 40, 19]
    cu, q, k, v, _ = make(docs, 2, 2, 8, seed=2)
    q[:] = 0
    o, lse = oracle.attn_fwd(q, k, v, cu, 0.125)
    for e in range(len(docs)):
        for t in range(cu[e], cu[e + 1]):
            cnt = t - cu[e] + 1
            np.testing.assert_allclose(lse[t], np.log(cnt), rtol=1e-14, atol=1e-15)
            np.testing.assert_allclose(o[t], v[cu[e]:t + 1].astype(np.float64).mean(axis=0), rtol=1e-13, atol=1e-15)


def test_p7_first_row_of_each_document():
    docs = [1, 9, 1, 1, 12]
    cu, q, k, v, do = make(docs, 4, 2, 8, seed=8)
    scale = 0.4
    o, lse = oracle.attn_fwd(q, k, v, cu, scale)
    dq = oracle.attn_bwd_dq(q, k, v, do, cu, scale)
    for e in range(len(docs)):
        t = cu[e]
        for h in range(4):
            np.testing.assert_allclose(o[t, h], v[t, h // 2].astype(np.float64), rtol=1e-15)
            np.testing.assert_allclose(lse[t, h], scale * np.dot(q[t, h].astype(np.float64), k[t, h // 2].astype(np.float64)), rtol=1e-14)
        np.testing.assert_allclose(dq[t], 0.0, atol=1e-15)
    # a length-1 document: dK = 0, dV = sum over the group's heads of dO
    dk, dv = oracle.attn_bwd_dkv(q, k, v, do, cu, scale)
    for e, L in enumerate(docs):
        if L == 1:
            t = cu[e]
            np.testing.assert_allclose(dk[t], 0.0, atol=1e-15)
            np.testing.assert_allclose(dv[t, 0], do[t, 0:2].astype(np.float64).sum(axis=0), rtol=1e-14)


def test_p8_poison_other_documents_and_the_future():
    docs = [14, 22, 9]
    cu, q, k, v, _ = make(docs, 2, 2, 8, seed=9)
    o, lse = oracle.attn_fwd(q, k, v, cu, 0.3)
    for e in range(len(docs)):
        a, b = cu[e], cu[e + 1]
        k2, v2 = k.copy(), v.copy()
        k2[:a] = 96.0; k2[b:] = -96.0; v2[:a] = 1e4; v2[b:] = -1e4
        o2, lse2 = oracle.attn_fwd(q, k2, v2, cu, 0.3)
        np.testing.assert_array_equal(o2[a:b], o[a:b]); np.testing.assert_array_equal(lse2[a:b], lse[a:b])
    t = 20                                       # future positions inside the same document
    k2, v2 = k.copy(), v.copy(); k2[t + 1:] = 64.0; v2[t + 1:] = 1e4
    o2, lse2 = oracle.attn_fwd(q, k2, v2, cu, 0.3, np.array([t]))
    np.testing.assert_array_equal(o2[0], o[t]); np.testing.assert_array_equal(lse2[0], lse[t])


def test_p9_adjoint_identity_for_dv():
    cu, q, k, v, do = make([10, 30, 8], 4, 2, 8, seed=10)
    scale = 0.35
    _, dv = oracle.attn_bwd_dkv(q, k, v, do, cu, scale)
    dV = bf16_exact(np.random.default_rng(5).standard_normal(v.shape))
    o_lin, _ = oracle.attn_fwd(q, k, dV, cu, scale)         # O is linear in V
    lhs = float((do.astype(np.float64) * o_lin).sum())
    rhs = float((dv * dV.astype(np.float64)).sum())
    assert abs(lhs - rhs) <= 1e-11 * max(1.0, abs(lhs))


def test_p10_key_shift_invariance():
    docs = [12, 21]
    cu, q, k, v, _ = make(docs, 2, 1, 8, seed=12)
    scale = 0.25
    o, lse = oracle.attn_fwd(q, k, v, cu, scale)
    c = bf16_exact(np.random.default_rng(3).standard_normal(8) * 0.5)
    k2 = k.copy(); k2[cu[1]:cu[2], 0] += c                   # exact in fp32 (bf16 + bf16)
    o2, lse2 = oracle.attn_fwd(q, k2, v, cu, scale)
    np.testing.assert_allclose(o2, o, rtol=1e-11, atol=1e-13)
    shift = scale * (q[cu[1]:cu[2]].astype(np.float64) @ c.astype(np.float64))
    np.testing.assert_allclose(lse2[cu[1]:cu[2]] - lse[cu[1]:cu[2]], shift, rtol=1e-11, atol=1e-12)
    np.testing.assert_array_equal(lse2[:cu[1]], lse[:cu[1]])


def test_merge_identity_commutes_and_matches_logsumexp():
    from scipy.special import logsumexp
    rng = np.random.default_rng(0)
    n, d = 9, 5
    oa, ob = rng.standard_normal((n, d)), rng.standard_normal((n, d))
    la, lb = rng.standard_normal(n) * 5, rng.standard_normal(n) * 5
    o, l = oracle.lse_merge(oa, la, ob, lb)
    np.testing.assert_allclose(l, logsumexp(np.stack([la, lb]), axis=0), rtol=1e-14)
    w = np.exp(la - l)[:, None]
    np.testing.assert_allclose(o, w * oa + (1 - w) * ob, rtol=1e-12, atol=1e-14)   # weights sum to 1
    o2, l2 = oracle.lse_merge(ob, lb, oa, la)
    np.testing.assert_allclose(o2, o, rtol=1e-14); np.testing.assert_allclose(l2, l, rtol=1e-15)
    ninf = np.full(n, -np.inf)
    o3, l3 = oracle.lse_merge(oa, la, np.zeros((n, d)), ninf)                       # identity element
    np.testing.assert_array_equal(o3, oa); np.testing.assert_array_equal(l3, la)
    o4, l4 = oracle.lse_merge(np.zeros((n, d)), ninf, np.zeros((n, d)), ninf)
    assert np.all(l4 == -np.inf) and np.all(o4 == 0) and not np.isnan(o4).any()


def test_partial_rows_without_keys_are_empty():
    cu, q, k, v, _ = make([6, 10], 2, 2, 4, seed=1)
    # rows 8..16 (second doc + tail) against keys 0..6 (first doc only): nothing visible
    o, lse = oracle.attn_partial(q, k, v, cu, 0.5, 8, 16, 0, 6)
    assert np.all(lse == -np.inf) and np.all(o == 0)


def test_p1_sparse_dout_rows_match_brute_force():
    # rows with dO = 0 are skipped by the oracle's dK/dV (they add exactly zero): same result as the full matrix form
    cu, q, k, v, do = make([9, 14, 1, 8], 4, 2, 8, seed=3)
    keep = np.zeros(len(q), dtype=bool); keep[[0, 5, 8, 9, 20, 22, 23, 31]] = True
    do = np.where(keep[:, None, None], do, np.float32(0))
    scale = 0.3
    _, _, dQ, dK, dV = brute(q, k, v, cu, scale, do)
    dk, dv = oracle.attn_bwd_dkv(q, k, v, do, cu, scale)
    assert np.abs(dk - dK).max() < 1e-12 and np.abs(dv - dV).max() < 1e-12
    cols = [0, 3, 9, 10, 22, 23, 24, 31]
    dk2, dv2 = oracle.attn_bwd_dkv(q, k, v, do, cu, scale, cols=cols)
    assert np.abs(dk2 - dK[cols]).max() < 1e-12 and np.abs(dv2 - dV[cols]).max() < 1e-12
    assert np.abs(oracle.attn_bwd_dq(q, k, v, do, cu, scale) - dQ).max() < 1e-12
