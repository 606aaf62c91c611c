"""ctypes front-end of the fp64 CPU oracle (oracle/sap_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import this.  It imports nothing
from paper_2606_30460_b200 (the CUDA path) and shares no code with it.

Parity status: every float function and plan() are pinned (tests/test_oracle_*.py); schedule() (compile Steps 2-3)
and codegen() (jitted code generation) are PARTIALLY PINNED - validity, closed forms, bounds, send/recv pairing and
the replay test are pinned; the choice among valid schedules and the stage offsets are a reading (R-5; the
paper's Fig. 3 is missing).

Arrays are numpy; Q/K/V/dO are float32 arrays holding bf16-exact values
(`tensor.float().numpy()`); every result is float64.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sap_oracle.cpp")
_LIB = os.path.join(_HERE, "libsap_oracle.so")

SKIP, FULL, DIAG = 0, 1, 2
ITEM_FIELDS = ("q_chunk", "kv_chunk", "doc_lo", "doc_hi", "mask_kind", "step",
               "q_begin", "q_end", "kv_begin", "kv_end")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (x86-64-v3 so the .so also runs on the GPU box's host)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O3", "-march=x86-64-v3", "-std=c++17", "-fopenmp", "-fPIC", "-shared",
               "-fno-fast-math", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.sap_oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(lib().sap_oracle_num_threads())


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(ctypes.c_void_p)


def _i32(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(ctypes.c_void_p)


def _i64_or_null(a):
    if a is None:
        return None, ctypes.c_void_p(0), 0
    a = np.ascontiguousarray(a, dtype=np.int64)
    return a, a.ctypes.data_as(ctypes.c_void_p), a.shape[0]


def _dims(q, k):
    N, Hq, d = q.shape
    Hkv = k.shape[1]
    return N, Hq, Hkv, d


def attn_fwd(q, k, v, cu_seqlens, scale: float, rows: Optional[Sequence[int]] = None):
    """Exact per-document causal attention.  Returns (O [n_rows,Hq,d], LSE [n_rows,Hq])."""
    q, qp = _f32(q); k, kp = _f32(k); v, vp = _f32(v)
    cu, cup = _i32(cu_seqlens)
    N, Hq, Hkv, d = _dims(q, k)
    rows_a, rp, nr = _i64_or_null(rows)
    if rows is None:
        nr = N
    o = np.empty((nr, Hq, d), dtype=np.float64)
    lse = np.empty((nr, Hq), dtype=np.float64)
    rc = lib().sap_oracle_fwd(qp, kp, vp, cup, ctypes.c_int(len(cu) - 1), ctypes.c_int64(N),
                              ctypes.c_int(Hq), ctypes.c_int(Hkv), ctypes.c_int(d),
                              ctypes.c_double(scale), rp, ctypes.c_int64(nr),
                              o.ctypes.data_as(ctypes.c_void_p), lse.ctypes.data_as(ctypes.c_void_p))
    if rc != 0:
        raise ValueError(f"sap_oracle_fwd: bad arguments ({rc})")
    return o, lse


def attn_partial(q, k, v, cu_seqlens, scale: float, q_begin: int, q_end: int, kv_begin: int, kv_end: int):
    """Partial attention of one work item.  Returns (O [rows,Hq,d], LSE [rows,Hq]); -inf/0 for empty rows."""
    q, qp = _f32(q); k, kp = _f32(k); v, vp = _f32(v)
    cu, cup = _i32(cu_seqlens)
    N, Hq, Hkv, d = _dims(q, k)
    nr = q_end - q_begin
    o = np.empty((nr, Hq, d), dtype=np.float64)
    lse = np.empty((nr, Hq), dtype=np.float64)
    rc = lib().sap_oracle_partial(qp, kp, vp, cup, ctypes.c_int(len(cu) - 1), ctypes.c_int64(N),
                                  ctypes.c_int(Hq), ctypes.c_int(Hkv), ctypes.c_int(d),
                                  ctypes.c_double(scale), ctypes.c_int64(q_begin), ctypes.c_int64(q_end),
                                  ctypes.c_int64(kv_begin), ctypes.c_int64(kv_end),
                                  o.ctypes.data_as(ctypes.c_void_p), lse.ctypes.data_as(ctypes.c_void_p))
    if rc != 0:
        raise ValueError("sap_oracle_partial: bad arguments")
    return o, lse


def lse_merge(o_a, lse_a, o_b, lse_b):
    """Exact merge of two partials over disjoint key sets.  o_* [...,d], lse_* [...]."""
    o_a = np.ascontiguousarray(o_a, dtype=np.float64); o_b = np.ascontiguousarray(o_b, dtype=np.float64)
    lse_a = np.ascontiguousarray(lse_a, dtype=np.float64); lse_b = np.ascontiguousarray(lse_b, dtype=np.float64)
    d = o_a.shape[-1]
    n = lse_a.size
    o = np.empty_like(o_a); lse = np.empty_like(lse_a)
    lib().sap_oracle_merge(o_a.ctypes.data_as(ctypes.c_void_p), lse_a.ctypes.data_as(ctypes.c_void_p),
                           o_b.ctypes.data_as(ctypes.c_void_p), lse_b.ctypes.data_as(ctypes.c_void_p),
                           ctypes.c_int64(n), ctypes.c_int(d),
                           o.ctypes.data_as(ctypes.c_void_p), lse.ctypes.data_as(ctypes.c_void_p))
    return o, lse


def attn_bwd_dq(q, k, v, dout, cu_seqlens, scale: float, rows: Optional[Sequence[int]] = None):
    q, qp = _f32(q); k, kp = _f32(k); v, vp = _f32(v); dout, dp = _f32(dout)
    cu, cup = _i32(cu_seqlens)
    N, Hq, Hkv, d = _dims(q, k)
    rows_a, rp, nr = _i64_or_null(rows)
    if rows is None:
        nr = N
    dq = np.empty((nr, Hq, d), dtype=np.float64)
    rc = lib().sap_oracle_bwd_dq(qp, kp, vp, dp, cup, ctypes.c_int(len(cu) - 1), ctypes.c_int64(N),
                                 ctypes.c_int(Hq), ctypes.c_int(Hkv), ctypes.c_int(d),
                                 ctypes.c_double(scale), rp, ctypes.c_int64(nr),
                                 dq.ctypes.data_as(ctypes.c_void_p))
    if rc != 0:
        raise ValueError("sap_oracle_bwd_dq: bad arguments")
    return dq


def attn_bwd_dkv(q, k, v, dout, cu_seqlens, scale: float, cols: Optional[Sequence[int]] = None):
    q, qp = _f32(q); k, kp = _f32(k); v, vp = _f32(v); dout, dp = _f32(dout)
    cu, cup = _i32(cu_seqlens)
    N, Hq, Hkv, d = _dims(q, k)
    cols_a, cp, nc = _i64_or_null(cols)
    if cols is None:
        nc = N
    dk = np.empty((nc, Hkv, d), dtype=np.float64)
    dv = np.empty((nc, Hkv, d), dtype=np.float64)
    rc = lib().sap_oracle_bwd_dkv(qp, kp, vp, dp, cup, ctypes.c_int(len(cu) - 1), ctypes.c_int64(N),
                                  ctypes.c_int(Hq), ctypes.c_int(Hkv), ctypes.c_int(d),
                                  ctypes.c_double(scale), cp, ctypes.c_int64(nc),
                                  dk.ctypes.data_as(ctypes.c_void_p), dv.ctypes.data_as(ctypes.c_void_p))
    if rc != 0:
        raise ValueError("sap_oracle_bwd_dkv: bad arguments")
    return dk, dv


class Plan:
    """Result of the brute-definition planner."""

    def __init__(self, items, chunk_offsets, kv_offsets, kv_index, kind_map):
        self.items = items                  # int32 [n_items, 10]
        self.chunk_offsets = chunk_offsets  # int32 [P+1]
        self.kv_offsets = kv_offsets        # int32 [P+1]
        self.kv_index = kv_index            # int32 [n_items]
        self.kind_map = kind_map            # uint8 [P, P]

    @property
    def n_items(self):
        return self.items.shape[0]


def plan(cu_seqlens, n_chunks: int) -> Plan:
    cu, cup = _i32(cu_seqlens)
    P = int(n_chunks)
    cap = max(1, P * (P + 1) // 2)
    items = np.zeros((cap, 10), dtype=np.int32)
    co = np.zeros(P + 1, dtype=np.int32)
    ko = np.zeros(P + 1, dtype=np.int32)
    ki = np.zeros(cap, dtype=np.int32)
    km = np.zeros((P, P), dtype=np.uint8) if P > 0 else np.zeros((0, 0), dtype=np.uint8)
    n = lib().sap_oracle_plan(cup, ctypes.c_int(len(cu) - 1), ctypes.c_int(P),
                              items.ctypes.data_as(ctypes.c_void_p), co.ctypes.data_as(ctypes.c_void_p),
                              ko.ctypes.data_as(ctypes.c_void_p), ki.ctypes.data_as(ctypes.c_void_p),
                              km.ctypes.data_as(ctypes.c_void_p))
    if n < 0:
        raise ValueError({-1: "invalid argument", -2: "bad cu_seqlens", -3: "N not divisible by n_chunks"}[n])
    return Plan(items[:n].copy(), co, ko, ki[:n].copy(), km)


def schedule(cu_seqlens, n_chunks: int, policy: int = 1):
    """Compile Steps 2-3, written out step by step in plain Python from the reading in DESIGN.md
    (R-5; the paper's Fig. 3 is missing).  Returns (slots int32 [n_items, 2] = (rank, stage), n_stages).

    policy 0: plain ring (:59): item (i, j) on rank i at stage i - j.
    policy 1: Step 2 per causal region (a document spanning chunks a..b, m = b - a + 1): diagonal items on their own
    rank at stage 0; a FULL item (i, j) stays on rank i at regional stage i - j if i - j <= m // 2, else the early
    rank j computes it at regional stage m - (i - j) (LightSeq-style balancing, :116).  Step 3: every rank runs at
    most one item per stage: it runs its items back to back in order of (regional stage, i, j), stage = position
    in that list (:118; shards travel point to point, so any order is legal); before that, Step 3a moves items off the busiest rank while
    that lowers its load ("striving to balance the computation load across all SAP ranks globally", :118).
    PARITY: pinned by validity (every item once, rank in {i, j}, one item per rank and stage), by the closed form
    for one document (floor(P/2) + 1 stages, loads within 1) and by makespan bounds; the choice among valid
    schedules is this reading's, not the paper's (figure missing) - "partially pinned".
    """
    pl = plan(cu_seqlens, n_chunks)
    cu = [int(x) for x in cu_seqlens]
    P = int(n_chunks)
    n = cu[-1] // P
    items = [tuple(int(v) for v in row) for row in pl.items]
    slots = np.zeros((len(items), 2), dtype=np.int32)
    if policy == 0:
        for x, it in enumerate(items):
            slots[x] = (it[0], it[0] - it[1])
        return slots, (int(slots[:, 1].max()) + 1 if len(items) else 0)
    regional = []
    for x, it in enumerate(items):
        i, j, doc_lo, kind = it[0], it[1], it[2], it[4]
        if kind == DIAG:
            slots[x, 0] = i
            regional.append(0)
            continue
        a, b = cu[doc_lo] // n, (cu[doc_lo + 1] - 1) // n          # chunks the region's document spans
        m, t = b - a + 1, i - j
        if t <= m // 2:
            slots[x, 0] = i
            regional.append(t)
        else:
            slots[x, 0] = j
            regional.append(m - t)
    # Step 3a: global balance - while the busiest rank (lowest index on ties) holds a FULL item whose other end
    # (the rank of its Q or of its K/V) has at least two items fewer, hand over the item whose other end is least
    # loaded (lowest item index on ties); its regional stage becomes t on rank i, m - t on rank j.
    load = [0] * P
    for x in range(len(items)):
        load[slots[x, 0]] += 1
    while True:
        R = max(range(P), key=lambda r: (load[r], -r))
        cands = [x for x in range(len(items)) if slots[x, 0] == R and items[x][4] != DIAG]
        if not cands:
            break
        other = lambda x: items[x][1] if R == items[x][0] else items[x][0]
        x = min(cands, key=lambda x: (load[other(x)], x))
        o = other(x)
        if load[o] + 1 >= load[R]:
            break
        load[R] -= 1
        load[o] += 1
        slots[x, 0] = o
        i, j, doc_lo = items[x][0], items[x][1], items[x][2]
        m, t = (cu[doc_lo + 1] - 1) // n - cu[doc_lo] // n + 1, i - j
        regional[x] = t if o == i else m - t
    # Step 3b: stages
    nxt = [0] * P
    for x in sorted(range(len(items)), key=lambda x: (regional[x], items[x][0], items[x][1])):
        slots[x, 1] = nxt[slots[x, 0]]          # a rank runs its items back to back in this order
        nxt[slots[x, 0]] += 1
    return slots, (int(slots[:, 1].max()) + 1 if len(items) else 0)


OP_SEND, OP_RECV, OP_COMPUTING, OP_COPY = 0, 1, 2, 3
T_Q, T_KV, T_O = 0, 1, 2


def codegen(cu_seqlens, n_chunks: int, slots, rank: int):
    """Jitted code generation for the forward pass (Table 1 :85-98), written out rule by rule.
    Codes are (stage, opcode, tensor, peer, item).  For every plan item (i, j) with slot (R, st):
      R runs `computing item` at stage st;
      if i != j and R == i: kv travels j -> i at stage st-1 (send on j, recv + copy on i);
      if i != j and R == j: q travels i -> j at stage st-1 (send on i, recv + copy on j) and the partial result o
                            travels j -> i at stage st+1 (send on j, recv + copy-and-rescale on i).
    Order inside a stage: SEND/RECV by (opcode, tensor, peer, item), then COMPUTING, then COPY by (tensor, peer, item).
    PARITY: the transport rules above are the paper's (who needs which tensor follows from where the block runs);
    the stage offsets (-1 / +1) and the order inside a stage are this build's reading - partially pinned: pinned by
    the executor test (every rank's replay reproduces the unchunked attention) and by send/recv pairing."""
    pl = plan(cu_seqlens, n_chunks)
    out = []
    for x, row in enumerate(pl.items):
        i, j = int(row[0]), int(row[1])
        R, st = int(slots[x][0]), int(slots[x][1])
        if R == rank:
            out.append((st, OP_COMPUTING, -1, -1, x))
        if i == j:
            continue
        if R == i:
            if rank == j:
                out.append((st - 1, OP_SEND, T_KV, i, x))
            if rank == i:
                out += [(st - 1, OP_RECV, T_KV, j, x), (st - 1, OP_COPY, T_KV, j, x)]
        else:
            if rank == i:
                out += [(st - 1, OP_SEND, T_Q, j, x), (st + 1, OP_RECV, T_O, j, x), (st + 1, OP_COPY, T_O, j, x)]
            if rank == j:
                out += [(st - 1, OP_RECV, T_Q, i, x), (st - 1, OP_COPY, T_Q, i, x), (st + 1, OP_SEND, T_O, i, x)]
    phase = {OP_SEND: 0, OP_RECV: 0, OP_COMPUTING: 1, OP_COPY: 2}
    out.sort(key=lambda c: (c[0], phase[c[1]], c[1] if phase[c[1]] == 0 else 0, c[2], c[3], c[4]))
    return np.array(out, dtype=np.int32).reshape(-1, 5)


T_DO, T_DQ, T_DKV = 3, 4, 5


def codegen_bwd(cu_seqlens, n_chunks: int, slots, rank: int):
    """Backward instruction list of `rank` (tensors do / dq / dkv of Table 1), rule by rule:
      R == i: kv travels j -> i at stage st-1, the dK/dV contribution (dkv) travels i -> j at stage st+1;
      R == j: q and do (with LSE, D) travel i -> j at stage st-1, the dQ contribution (dq) travels j -> i at st+1.
    Same format and order as codegen().  Partially pinned, as codegen()."""
    pl = plan(cu_seqlens, n_chunks)
    out = []

    def transfer(stage, tensor, src, dst, x):
        if rank == src:
            out.append((stage, OP_SEND, tensor, dst, x))
        if rank == dst:
            out.extend([(stage, OP_RECV, tensor, src, x), (stage, OP_COPY, tensor, src, x)])

    for x, row in enumerate(pl.items):
        i, j = int(row[0]), int(row[1])
        R, st = int(slots[x][0]), int(slots[x][1])
        if R == rank:
            out.append((st, OP_COMPUTING, -1, -1, x))
        if i == j:
            continue
        if R == i:
            transfer(st - 1, T_KV, j, i, x)
            transfer(st + 1, T_DKV, i, j, x)
        else:
            transfer(st - 1, T_Q, i, j, x)
            transfer(st - 1, T_DO, i, j, x)
            transfer(st + 1, T_DQ, j, i, x)
    phase = {OP_SEND: 0, OP_RECV: 0, OP_COMPUTING: 1, OP_COPY: 2}
    out.sort(key=lambda c: (c[0], phase[c[1]], c[1] if phase[c[1]] == 0 else 0, c[2], c[3], c[4]))
    return np.array(out, dtype=np.int32).reshape(-1, 5)


def attn_bwd_item(q, k, v, dout, lse, dsum, cu_seqlens, scale: float, q_begin: int, q_end: int, kv_begin: int,
                  kv_end: int):
    """Backward contribution of ONE work item (rows [q_begin,q_end) x keys [kv_begin,kv_end), document AND causal
    mask), given the row statistics of the COMPLETE forward: lse [N,Hq] and dsum = rowsum(dO*O) [N,Hq].
      P = exp(scale q.k - LSE) on visible pairs; dP = dO v^T; dS = P (dP - D);
      dQ_rows = scale dS k;  dK_keys = scale dS^T q (summed over the q-heads of a group);  dV_keys = P^T dO.
    Returns (dq [q_end-q_begin,Hq,d], dk, dv [kv_end-kv_begin,Hkv,d]) in fp64.  Plain matrix form (small inputs).
    Pinned by: the sum over all items of a plan equals attn_bwd_dq / attn_bwd_dkv (tests/test_executor_gloo.py)."""
    q = np.asarray(q, np.float64); k = np.asarray(k, np.float64); v = np.asarray(v, np.float64)
    dout = np.asarray(dout, np.float64)
    cu = np.asarray(cu_seqlens)
    N, Hq, d = q.shape
    Hkv = k.shape[1]
    g = Hq // Hkv
    rows = np.arange(q_begin, q_end); keys = np.arange(kv_begin, kv_end)
    doc_r = np.searchsorted(cu, rows, side="right") - 1
    doc_k = np.searchsorted(cu, keys, side="right") - 1
    vis = (doc_r[:, None] == doc_k[None, :]) & (keys[None, :] <= rows[:, None])
    dq = np.zeros((len(rows), Hq, d)); dk = np.zeros((len(keys), Hkv, d)); dv = np.zeros((len(keys), Hkv, d))
    for h in range(Hq):
        hk = h // g
        S = scale * q[rows, h] @ k[keys, hk].T
        P = np.where(vis, np.exp(S - lse[rows, h][:, None]), 0.0)
        dP = dout[rows, h] @ v[keys, hk].T
        dS = P * (dP - dsum[rows, h][:, None])
        dq[:, h] = scale * dS @ k[keys, hk]
        dk[:, hk] += scale * dS.T @ q[rows, h]
        dv[:, hk] += P.T @ dout[rows, h]
    return dq, dk, dv
