"""ctypes front-end of the fp64 CPU oracle (oracle/sap_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import this.  It imports nothing
from paper_2606_30460_b200 (the CUDA path) and shares no code with it.

Parity status: every float function and plan() are pinned (tests/test_oracle_*.py).  For the compile side of the
NEXT rows the oracle no longer mirrors the library: min_makespan() is the exhaustive definition of the best possible
makespan (pinned by closed forms) and check_codes() is a legality checker of instruction lists written from Table 1 and
PAPER.md:100-102,:120-124 (pinned by hand-made legal and illegal lists) - neither generates a schedule or a code list.
schedule() remains as the step-by-step restatement of the reading DESIGN.md R-5 (the paper's Fig. 3 is missing): it
pins that the library implements that reading, the reading itself is scored against min_makespan().

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
_LIB_OVERRIDE = os.environ.get("SAP_ORACLE_LIB")   # an instrumented build (ASan / UBSan run)

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
        _lib = ctypes.CDLL(_LIB_OVERRIDE or build())
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
    PARITY: this function restates the reading R-5; what pins the READING is min_makespan(): on every tiny layout
    (P <= 6, <= 3 documents) the makespan of this schedule is within one block of the exhaustive optimum, and equal
    to it for a single document (tests/test_schedule.py).
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


def min_makespan(cu_seqlens, n_chunks: int, limit: int = 1 << 22):
    """The smallest makespan, in block units, ANY assignment of plan items to ranks can reach (Steps
    2-3 decide "which rank computes each block" and "the stage index"; one block per rank and stage): every DIAG item
    runs on its own rank, every FULL item (i, j) on rank i (K/V_j travels) or on rank j (Q_i travels, the partial
    travels back); a rank runs its items back to back, so the makespan is the largest number of items on one rank.
    Exhaustive over the 2^(#FULL) assignments - the definition, no heuristic; tiny inputs only."""
    pl = plan(cu_seqlens, n_chunks)
    P = int(n_chunks)
    load0 = [0] * P
    full = []
    for row in pl.items:
        i, j, kind = int(row[0]), int(row[1]), int(row[4])
        if kind == DIAG:
            load0[i] += 1
        else:
            full.append((i, j))
    if (1 << len(full)) > limit:
        raise ValueError("too many FULL items for the exhaustive search")
    best = None
    for mask in range(1 << len(full)):
        load = list(load0)
        for b, (i, j) in enumerate(full):
            load[j if (mask >> b) & 1 else i] += 1
        m = max(load)
        best = m if best is None or m < best else best
    return best if best is not None else 0


OP_SEND, OP_RECV, OP_COMPUTING, OP_COPY = 0, 1, 2, 3
T_Q, T_KV, T_O, T_DO, T_DQ, T_DKV = 0, 1, 2, 3, 4, 5


def check_codes(cu_seqlens, n_chunks: int, slots, code_lists, backward: bool = False):
    """Legality of the instruction lists of ALL ranks (code_lists[r] = int array [n, 5] of (stage, opcode, tensor, peer,
    item)) for a schedule `slots` - a checker, not a generator: any list that passes can be executed, whatever stage
    offsets or in-stage order its author chose.  Returns a list of violations (empty = legal).  Rules, each from the
    paper's description of the execute side (Table 1):

      R1  a rank walks its list stage by stage; inside a stage the SEND / RECV codes come first (one batched
          isend/irecv, in flight while the block is computed, :122-124), then COMPUTING, then COPY (:102).
      R2  every plan item is computed exactly once, by the rank and at the stage its slot names, and a rank computes at
          most one item per stage (:116-118).
      R3  operands are in the compute buffer before COMPUTING: an item (i, j) computed on rank R != i needs q of chunk i
          (and, backward, do) - RECV from i and COPY at a stage EARLIER than the computing stage; R != j needs kv of
          chunk j the same way.  A rank never receives a tensor it owns or does not need ("trim redundant
          communication", :106).
      R4  every SEND has its RECV with the same (stage, tensor, item) on the peer and vice versa ("send/recv pairs
          aligned", :124), sent by the rank that owns / produced the tensor; every RECV has its COPY in the same or a
          later stage on the same rank.
      R5  what a rank computes for another is returned AFTER it exists: forward, R != i sends the partial o to i at a
          stage LATER than the computing stage; backward, R != i returns dq to i and R != j returns dkv to j.  Nothing
          else travels.
    """
    pl = plan(cu_seqlens, n_chunks)
    P = int(n_chunks)
    items = [(int(r[0]), int(r[1])) for r in pl.items]
    bad = []
    sends, recvs, copies, computes = {}, {}, {}, {}
    phase = {OP_SEND: 0, OP_RECV: 0, OP_COMPUTING: 1, OP_COPY: 2}
    for r in range(P):
        last = None
        per_stage = {}
        for st, op, tensor, peer, item in (tuple(int(v) for v in c) for c in code_lists[r]):
            key = (st, phase.get(op, 9))
            if last is not None and key < last:
                bad.append(f"R1 rank {r}: code (stage {st}, opcode {op}) is out of order")
            last = key
            if not 0 <= item < len(items):
                bad.append(f"rank {r}: item {item} does not exist"); continue
            if op == OP_COMPUTING:
                if item in computes:
                    bad.append(f"R2 item {item} computed twice")
                computes[item] = (r, st)
                per_stage[st] = per_stage.get(st, 0) + 1
                if per_stage[st] > 1:
                    bad.append(f"R2 rank {r} computes two items at stage {st}")
            elif op == OP_SEND:
                if (tensor, r, peer, item) in sends: bad.append(f"R4 duplicate SEND {(tensor, r, peer, item)}")
                sends[(tensor, r, peer, item)] = st
            elif op == OP_RECV:
                if (tensor, peer, r, item) in recvs: bad.append(f"R4 duplicate RECV {(tensor, peer, r, item)}")
                recvs[(tensor, peer, r, item)] = st
            elif op == OP_COPY:
                copies[(tensor, peer, r, item)] = st
            else:
                bad.append(f"rank {r}: unknown opcode {op}")
    for x, (i, j) in enumerate(items):
        R, st = int(slots[x][0]), int(slots[x][1])
        if computes.get(x) != (R, st):
            bad.append(f"R2 item {x} computed at {computes.get(x)}, its slot says {(R, st)}")
    if set(sends) != set(recvs):
        bad.append(f"R4 unpaired SEND / RECV: {sorted(set(sends) ^ set(recvs))[:4]}")
    for key in set(sends) & set(recvs):
        if sends[key] != recvs[key]:
            bad.append(f"R4 SEND at stage {sends[key]} but RECV at stage {recvs[key]} for {key}")
        if key not in copies or copies[key] < recvs[key]:
            bad.append(f"R4 RECV {key} has no COPY in the same or a later stage")
    if set(copies) - set(recvs):
        bad.append(f"R4 COPY without RECV: {sorted(set(copies) - set(recvs))[:4]}")
    need = set()          # every transfer the schedule requires, as (tensor, src, dst, item) with its stage constraint
    for x, (i, j) in enumerate(items):
        R, st = int(slots[x][0]), int(slots[x][1])
        ops_in = []
        if R != i:
            ops_in += [(T_Q, i)] + ([(T_DO, i)] if backward else [])
        if R != j:
            ops_in += [(T_KV, j)]
        for tensor, src in ops_in:                                    # R3
            key = (tensor, src, R, x)
            need.add(key)
            if key not in copies:
                bad.append(f"R3 item {x} on rank {R}: tensor {tensor} of chunk {src} never arrives")
            elif copies[key] >= st:
                bad.append(f"R3 item {x} computed at stage {st} but tensor {tensor} is copied at stage {copies[key]}")
        outs = []
        if R != i:
            outs.append((T_DQ if backward else T_O, i))
        if backward and R != j:
            outs.append((T_DKV, j))
        for tensor, dst in outs:                                      # R5
            key = (tensor, R, dst, x)
            need.add(key)
            if key not in sends:
                bad.append(f"R5 item {x}: result tensor {tensor} is never returned to rank {dst}")
            elif sends[key] <= st:
                bad.append(f"R5 item {x} computed at stage {st} but its result is sent at stage {sends[key]}")
    if set(sends) - need:
        bad.append(f"R3/R5 transfers nobody needs: {sorted(set(sends) - need)[:4]}")
    return bad


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
