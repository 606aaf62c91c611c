"""SAP ranks driven from ONE process over stitched tensors (the B200-native exchange).

The paper's ranks exchange K/V (and dK/dV, dQ) shards with grouped send / recv around a FlashAttention call
(PAPER.md:59, :100-102, :124).  Inside an NVLink / NVSwitch domain nothing has to be shipped ahead of the kernel: every
[N, H, d] tensor lives in one stitched range (`api.Stitched`: chunk c = memory of the device that owns sequence chunk
c), all tensors keep global token indices, and rank c launches the library's kernels restricted to its own chunks on
its own device.  Its forward reads the K/V tiles its plan names where they live (TMA over NVLink), its KV-stationary
backward streams Q / dO the same way and adds its dQ contributions into the owner's fp32 accumulator (red.global) -
transfer and compute are one kernel, and the chunk pairs the plan skips move no byte.

Control flow = four phases with two group barriers (stream events; no kernel ever waits on another kernel):
    forward:  every rank: sap_attn_fwd_chunks(own q-chunk)
    backward: every rank: sap_attn_bwd_begin(own rows: D, zeroed accumulator)   | barrier: all D written, all rows zeroed
              every rank: sap_attn_bwd_chunks(own K/V chunk)                     | barrier: all contributions added
              every rank: sap_attn_bwd_end(own dQ rows)
Ranks that share a device share its stream (their launches run one after the other): with every chunk on device 0 this
is the one-GPU emulation the tests run; with distinct P2P-capable devices it is the multi-GPU form - not run anywhere
yet (no box with a second GPU), so treat that path as untested.  `RankGroup` drives all devices from one process;
`ProcessRank` is the one-process-per-GPU form (the stitched ranges are assembled from chunks the processes export to
one another, the barriers are group barriers): tested with two processes on the one GPU of the box.
"""
from __future__ import annotations

from typing import Dict, List, Optional, Sequence

from . import api


def workspace_units(n_tokens: int, n_chunks: int, n_q_heads: int, head_dim: int, granularity: int):
    """Layout of the backward workspace (sap_workspace_bytes: D fp32 [Hq, N] padded to 256 B, then the fp32 dQ accumulator
    [N, Hq, d]) as equal units of a stitched range, so that the accumulator rows of chunk c can live with the owner of
    chunk c - the dQ contributions of every rank (red.global) then land in the memory of the rank that will read them,
    not in one rank's.  Returns (unit_bytes, units_per_chunk) with unit 0 = the D array, or None when the sizes do not
    line up (D not a multiple of the allocation granularity, or a chunk's accumulator not a multiple of D)."""
    d_bytes = (n_tokens * n_q_heads * 4 + 255) // 256 * 256
    acc_chunk = (n_tokens // n_chunks) * n_q_heads * head_dim * 4
    if d_bytes % granularity != 0 or acc_chunk % d_bytes != 0:
        return None
    return d_bytes, acc_chunk // d_bytes


class RankGroup:
    def __init__(self, cu_seqlens: Sequence[int], n_chunks: int, devices: Optional[Sequence[int]] = None):
        import torch
        self.P = int(n_chunks)
        self.devices: List[int] = [0] * self.P if devices is None else [int(d) for d in devices]
        if len(self.devices) != self.P:
            raise ValueError("one device per chunk")
        self.cu_seqlens = list(cu_seqlens)
        self.n_tokens = int(self.cu_seqlens[-1])
        self.plans: Dict[int, api.Plan] = {}
        self.cu_dev = {}
        self.streams = {}
        for dev in sorted(set(self.devices)):          # a plan's device mirror lives on one device: one plan per device
            with torch.cuda.device(dev):
                plan = api.sap_plan(self.cu_seqlens, self.P)
                plan.upload()
                self.plans[dev] = plan
                self.cu_dev[dev] = plan.cu_seqlens_dev(torch.device("cuda", dev))
                self.streams[dev] = torch.cuda.Stream(device=dev)
        self._keep = []

    # ------------------------------------------------------------------ memory
    def tensor(self, tail_shape: Sequence[int], dtype):
        """[N, *tail_shape] in a stitched range: rows of chunk c in the memory of devices[c]."""
        import torch
        n = self.n_tokens // self.P
        row = 1
        for x in tail_shape:
            row *= int(x)
        chunk_bytes = n * row * torch.empty((), dtype=dtype).element_size()
        s = api.Stitched(self.P, chunk_bytes, self.devices, sorted(set(self.devices)))
        return s.tensor((self.n_tokens, *tail_shape), dtype)

    def shared(self, shape: Sequence[int], dtype):
        """An array every rank reads and writes rows of but that cannot be split by chunk ([Hq, N] LSE, the backward
        workspace): one allocation on the first device, mapped for all of them."""
        import torch
        nbytes = torch.empty((), dtype=dtype).element_size()
        for x in shape:
            nbytes *= int(x)
        g = api.Stitched.granularity(self.devices[0])
        s = api.Stitched(1, (nbytes + g - 1) // g * g, [self.devices[0]], sorted(set(self.devices)))
        return s.tensor(tuple(shape), dtype)

    def workspace(self, n_q_heads: int, n_kv_heads: int, head_dim: int):
        """The backward workspace; the accumulator rows of chunk c on devices[c] when the sizes line up (workspace_units)."""
        import torch
        plan = self.plans[self.devices[0]]
        nbytes = api.sap_workspace_bytes(plan, n_q_heads, n_kv_heads, head_dim, api.SAP_PASS_BWD)
        lay = workspace_units(self.n_tokens, self.P, n_q_heads, head_dim, api.Stitched.granularity(self.devices[0]))
        if lay is None:
            return self.shared((nbytes,), torch.uint8)
        unit, per = lay
        owners = [self.devices[0]] + [self.devices[c] for c in range(self.P) for _ in range(per)]
        s = api.Stitched(len(owners), unit, owners, sorted(set(self.devices)))
        return s.tensor((nbytes,), torch.uint8)

    # ------------------------------------------------------------------ control
    def _fork(self):
        import torch
        for dev, st in self.streams.items():
            ev = torch.cuda.Event()
            with torch.cuda.device(self.devices[0]):
                ev.record(torch.cuda.current_stream())
            st.wait_event(ev)

    def _barrier(self):
        """Every rank's stream waits for the work every other rank's stream has been given so far."""
        import torch
        evs = []
        for dev, st in self.streams.items():
            ev = torch.cuda.Event()
            ev.record(st)
            evs.append(ev)
        for st in self.streams.values():
            for ev in evs:
                st.wait_event(ev)

    def _join(self):
        import torch
        cur = torch.cuda.current_stream(self.devices[0])
        for st in self.streams.values():
            ev = torch.cuda.Event()
            ev.record(st)
            cur.wait_event(ev)

    def _each_rank(self, fn):
        import torch
        for c, dev in enumerate(self.devices):
            with torch.cuda.device(dev):
                fn(c, self.plans[dev], self.cu_dev[dev], self.streams[dev])

    def forward(self, q, k, v, out, lse, softmax_scale: Optional[float] = None):
        self._fork()
        self._each_rank(lambda c, plan, cu, st: api.sap_attn_fwd_chunks(q, k, v, cu, plan, c, c + 1, out, lse,
                                                                        softmax_scale=softmax_scale, stream=st))
        self._join()

    def backward(self, dout, q, k, v, out, lse, dq, dk, dv, workspace, softmax_scale: Optional[float] = None):
        n_kv_heads = k.shape[1]
        self._fork()
        self._each_rank(lambda c, plan, cu, st: api.sap_attn_bwd_begin(dout, out, plan, c, c + 1, n_kv_heads, workspace, stream=st))
        self._barrier()        # every D written, every accumulator row zeroed
        self._each_rank(lambda c, plan, cu, st: api.sap_attn_bwd_chunks(dout, q, k, v, lse, cu, plan, c, c + 1, dk, dv, workspace,
                                                                        softmax_scale=softmax_scale, stream=st))
        self._barrier()        # every dQ contribution added
        self._each_rank(lambda c, plan, cu, st: api.sap_attn_bwd_end(plan, c, c + 1, dq, n_kv_heads, workspace,
                                                                     softmax_scale=softmax_scale, stream=st))
        self._join()


# ---------------------------------------------------------------------------------------------------------------------
# One process per GPU (the launch model of torch.distributed): the same phases, the barriers are group barriers of the
# process group, and the stitched ranges are assembled from chunks the processes export to one another.
_MAX_FDS_PER_MESSAGE = 253      # Linux SCM_MAX_FD: one sendmsg carries at most this many descriptors


def exchange_fds(rank: int, world: int, my_fds: Dict[int, int], group=None, tag: str = "sap") -> Dict[int, Dict[int, int]]:
    """Every rank hands the file descriptors `my_fds` (key -> fd, e.g. the exported chunks it owns) to every other
    rank: descriptors only travel between processes of one host over a Unix socket (SCM_RIGHTS).  Returns
    {sender rank: {key: fd valid in THIS process}}; the receiver closes them once imported.  Needs an initialised
    torch.distributed group (any backend: used for one broadcast and two barriers).

    The sockets live in a directory rank 0 creates for this exchange with mode 0700 (mkdtemp) and names to the others
    through the process group, so no other user can connect.  A message is accepted only from a process of this user
    (SO_PEERCRED), from a rank of the group that has not sent yet, and only whole: key count, payload length and the
    number of descriptors must agree and the ancillary data must not be truncated.  Anything else raises; descriptors
    received up to then are closed."""
    import array
    import os
    import shutil
    import socket
    import struct
    import tempfile
    import torch.distributed as dist

    if world == 1:
        return {}
    if len(my_fds) > _MAX_FDS_PER_MESSAGE:
        raise ValueError(f"at most {_MAX_FDS_PER_MESSAGE} descriptors per exchange, got {len(my_fds)}")
    box = [tempfile.mkdtemp(prefix=f"{tag}_fd_") if rank == 0 else None]
    dist.broadcast_object_list(box, src=0 if group is None else dist.get_global_rank(group, 0), group=group)
    root = box[0]
    path = os.path.join(root, str(rank))
    srv = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)
    got: Dict[int, Dict[int, int]] = {}

    def fail(why):
        for fds in got.values():
            for fd in fds.values():
                os.close(fd)
        raise RuntimeError(f"exchange_fds (rank {rank}): {why}")

    try:
        srv.bind(path)
        srv.listen(world)
        dist.barrier(group=group)                      # every rank listens
        keys = sorted(my_fds)
        for peer in range(world):                      # send to everybody (small messages: the connects do not block)
            if peer == rank:
                continue
            c = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)
            c.connect(os.path.join(root, str(peer)))
            payload = struct.pack(f"<ii{len(keys)}i", rank, len(keys), *keys)
            fds = array.array("i", [my_fds[k] for k in keys])
            c.sendmsg([payload], [(socket.SOL_SOCKET, socket.SCM_RIGHTS, fds)] if keys else [])
            c.close()
        for _ in range(world - 1):
            conn, _addr = srv.accept()
            try:
                _pid, uid, _gid = struct.unpack("3i", conn.getsockopt(socket.SOL_SOCKET, socket.SO_PEERCRED, struct.calcsize("3i")))
                msg, anc, flags, _a = conn.recvmsg(8 + 4 * _MAX_FDS_PER_MESSAGE, socket.CMSG_SPACE(4 * _MAX_FDS_PER_MESSAGE))
            finally:
                conn.close()
            fds = array.array("i")
            for level, typ, data in anc:
                if level == socket.SOL_SOCKET and typ == socket.SCM_RIGHTS:
                    fds.frombytes(data[: len(data) - (len(data) % fds.itemsize)])
            fds = list(fds)
            sender, n = struct.unpack_from("<ii", msg) if len(msg) >= 8 else (-1, -1)
            ok = (uid == os.getuid() and not (flags & (socket.MSG_CTRUNC | socket.MSG_TRUNC)) and 0 <= sender < world and
                  sender != rank and sender not in got and 0 <= n <= _MAX_FDS_PER_MESSAGE and len(msg) == 8 + 4 * n and len(fds) == n)
            if not ok:
                for fd in fds:
                    os.close(fd)
                fail(f"malformed or foreign message (uid {uid}, sender {sender}, {n} keys, {len(msg)} bytes, {len(fds)} descriptors, "
                     f"flags {flags:#x})")
            ks = struct.unpack_from(f"<{n}i", msg, 8)
            if len(set(ks)) != n:
                for fd in fds:
                    os.close(fd)
                fail(f"rank {sender} sent duplicate keys")
            got[sender] = dict(zip(ks, fds))
        dist.barrier(group=group)                      # every rank has received
    except BaseException:
        if rank == 0:                                  # nobody will reach the closing barrier: do not leave the directory behind
            shutil.rmtree(root, ignore_errors=True)
        raise
    finally:
        srv.close()
        if os.path.exists(path):
            os.unlink(path)
    dist.barrier(group=group)                          # every socket is gone: rank 0 removes the directory
    if rank == 0:
        shutil.rmtree(root, ignore_errors=True)
    return got


def launch_chunks(rank: int, world: int, n_chunks: int, balance: str = "zigzag") -> List[int]:
    """The chunks rank `rank` LAUNCHES (its q-chunks in the forward, its kv-chunks in the backward).  With stitched
    tensors that is independent of whose memory a chunk is, so the causal imbalance of contiguous ownership (the last
    rank's rows see every chunk, the first rank's only their own; the paper balances it by moving blocks between
    ranks) is removed by the assignment alone: "zigzag" gives rank r the chunks r, 2W-1-r, 2W+r, ...
    (a cheap chunk paired with an expensive one); "contiguous" = the chunks whose memory the rank owns."""
    per = n_chunks // world
    if balance == "contiguous":
        return list(range(rank * per, (rank + 1) * per))
    out = []
    for lap in range(per):
        out.append(lap * world + (rank if lap % 2 == 0 else world - 1 - rank))
    return out


def chunk_work(cu_seqlens: Sequence[int], n_chunks: int):
    """Visible (row, key) pairs per q-chunk (the rows of the chunk: what a forward launch on it computes) and per kv-chunk
    (the keys of the chunk: what a backward launch on it computes), from cu_seqlens alone: row t sees t - start(doc(t)) + 1
    keys, key s is seen by end(doc(s)) - s rows."""
    import numpy as np
    cu = np.asarray(cu_seqlens, dtype=np.int64)
    N = int(cu[-1])
    t = np.arange(N, dtype=np.int64)
    doc = np.searchsorted(cu, t, side="right") - 1
    n = N // n_chunks
    q_work = (t - cu[doc] + 1).reshape(n_chunks, n).sum(axis=1)
    kv_work = (cu[doc + 1] - t).reshape(n_chunks, n).sum(axis=1)
    return [int(x) for x in q_work], [int(x) for x in kv_work]


def assign_by_work(work: Sequence[int], world: int) -> List[List[int]]:
    """Longest-processing-time greedy: chunks in order of decreasing work (lower index first on ties), each to the rank
    with the least work so far (lowest rank on ties).  Deterministic: every rank computes the same assignment."""
    load = [0] * world
    out: List[List[int]] = [[] for _ in range(world)]
    for c in sorted(range(len(work)), key=lambda c: (-work[c], c)):
        r = min(range(world), key=lambda r: (load[r], r))
        out[r].append(c)
        load[r] += work[c]
    return [sorted(x) for x in out]


def link_bytes(cu_seqlens: Sequence[int], n_chunks: int, world: int, design: str, n_q_heads: int, n_kv_heads: int,
               head_dim: int) -> List[Dict[str, int]]:
    """Bytes each rank moves over NVLink in one forward + backward, counted from the tile programs the kernels walk
    (sap_debug_tile_program), with contiguous ownership (rank r owns and launches chunks [r P/W, (r+1) P/W)).  Host only.

    design "stitched" (RankGroup / ProcessRank): tensors are read where they live.  A rank's kernel loads every
        streamed tile it needs through TMA; a tile in a peer's memory is cached in the OWNER's L2, not the reader's, so
        each load of it crosses the link - the reuse that keeps the one-GPU DRAM traffic low turns into link traffic.
          forward  : per (Q tile, streamed 128-key tile, work item): K + V tile = 2 * 128 * d * 2 B; work items per tile =
                     Hq / 2 when Hq / Hkv is even (two q-heads of a group share the stream), Hq otherwise
          backward : per (K/V tile, streamed 128-row tile, q-head): Q + dO tile = 2 * 128 * d * 2 B plus LSE and D
                     (2 * 128 * 4 B) read, and 128 * d * 4 B of fp32 dQ contributions sent with red.global to the
                     owner of the rows (ranks.workspace_units keeps the accumulator rows with the chunk's owner)
    design "staged" (the paper's own exchange; executor.py / ring.py): every remote shard a
        rank needs travels ONCE into local staging and the kernels run on local memory.
          forward  : K_j, V_j rows [kv_begin, kv_end) of every remote chunk j some owned q-chunk has an item against
          backward : K/V-stationary at the owner of j: Q_i, dO_i (+ LSE, D) rows [q_begin, q_end) of every remote chunk
                     i, once, and one fp32 dQ partial of those rows sent back (Table 1 copy-dq, :95-98)
    Returns per rank {"fwd_read", "bwd_read", "bwd_red"} in bytes ("bwd_red": red.global traffic / dQ partials SENT).
    Tile rows past the end of a document are counted as loaded (the kernels load whole boxes)."""
    import numpy as np
    if design not in ("stitched", "staged"):
        raise ValueError("design is 'stitched' or 'staged'")
    if n_chunks % world != 0:
        raise ValueError("n_chunks must be a multiple of the number of ranks")
    plan = api.sap_plan(cu_seqlens, n_chunks)
    N, per = plan.n_tokens, n_chunks // world
    n = N // n_chunks
    owner = lambda t: min(t // n, n_chunks - 1) // per          # rank that owns token t
    Hq, Hkv, d = int(n_q_heads), int(n_kv_heads), int(head_dim)
    out = [{"fwd_read": 0, "bwd_read": 0, "bwd_red": 0} for _ in range(world)]
    if design == "staged":
        items = plan.items
        for r in range(world):
            mine = range(r * per, (r + 1) * per)
            kv_span: Dict[int, List[int]] = {}      # remote kv-chunk j -> [lo, hi) over the items of my q-chunks
            q_span: Dict[int, List[int]] = {}       # remote q-chunk i -> [lo, hi) over the items of my kv-chunks
            for i, j, _dl, _dh, _kind, _step, qb, qe, kb, ke in items.tolist():
                if i in mine and j not in mine:
                    sp = kv_span.setdefault(j, [kb, ke]); sp[0] = min(sp[0], kb); sp[1] = max(sp[1], ke)
                if j in mine and i not in mine:
                    sp = q_span.setdefault(i, [qb, qe]); sp[0] = min(sp[0], qb); sp[1] = max(sp[1], qe)
            out[r]["fwd_read"] = sum(hi - lo for lo, hi in kv_span.values()) * Hkv * d * 2 * 2
            rows = sum(hi - lo for lo, hi in q_span.values())
            out[r]["bwd_read"] = rows * Hq * (d * 2 * 2 + 2 * 4)
            out[r]["bwd_red"] = rows * Hq * d * 4
        return out
    share = 2 if (Hq // Hkv) % 2 == 0 else 1
    kv_kind = 7 if d == 128 else 6              # 256-key pair-tiles at head_dim 128, 128-key tiles otherwise
    for r in range(world):
        tiles, segs = plan.tile_program(5, r * per, (r + 1) * per)
        loads = 0
        for _row0, _rows, sb, se in tiles.tolist():
            for tb, te, *_ in segs[sb:se].tolist():
                loads += sum(1 for t in range(tb, te, 128) if owner(t) != r)
        out[r]["fwd_read"] = loads * (Hq // share) * 2 * 128 * d * 2
        tiles, segs = plan.tile_program(kv_kind, r * per, (r + 1) * per)
        loads = 0
        for _row0, _rows, sb, se in tiles.tolist():
            for tb, te, *_ in segs[sb:se].tolist():
                loads += sum(1 for t in range(tb, te, 128) if owner(t) != r)
        out[r]["bwd_read"] = loads * Hq * (2 * 128 * d * 2 + 2 * 128 * 4)
        out[r]["bwd_red"] = loads * Hq * 128 * d * 4
    return out


class ProcessRank:
    """This process = SAP rank `rank` of `world` on its own CUDA device.  The sequence has n_chunks chunks (a multiple of
    world; default one per rank); the rank OWNS the memory of a contiguous block of them and LAUNCHES the
    chunks the balance policy gives it: "work" (default) = by the visible pairs of each chunk, computed from cu_seqlens
    (the compile-time information of PAPER.md:106), separately for the forward (q-chunks) and the backward (kv-chunks);
    "zigzag" / "contiguous" = `launch_chunks`."""

    def __init__(self, cu_seqlens: Sequence[int], rank: int, world: int, device: int, group=None,
                 n_chunks: Optional[int] = None, balance: str = "work"):
        import torch
        self.rank, self.world, self.device, self.group = int(rank), int(world), int(device), group
        self.P = int(world if n_chunks is None else n_chunks)
        if self.P % self.world != 0:
            raise ValueError("n_chunks must be a multiple of the number of ranks")
        self.cu_seqlens = list(cu_seqlens)
        self.n_tokens = int(self.cu_seqlens[-1])
        torch.cuda.set_device(self.device)
        self.plan = api.sap_plan(self.cu_seqlens, self.P)
        self.plan.upload()
        self.cu_dev = self.plan.cu_seqlens_dev(torch.device("cuda", self.device))
        per = self.P // self.world
        self.owned = list(range(self.rank * per, (self.rank + 1) * per))
        if balance == "work":
            q_work, kv_work = chunk_work(self.cu_seqlens, self.P)
            self.launch = assign_by_work(q_work, self.world)[self.rank]        # forward, D pre-pass, dQ post pass: q-chunks
            self.launch_kv = assign_by_work(kv_work, self.world)[self.rank]    # backward main kernel: kv-chunks
        else:
            self.launch = launch_chunks(self.rank, self.world, self.P, balance)
            self.launch_kv = list(self.launch)
        self._n_ranges = 0

    def _assemble(self, n_chunks: int, chunk_bytes: int, own: Sequence[bool]) -> api.Stitched:
        import os
        s = api.Stitched.create_local(n_chunks, chunk_bytes, self.device, own)
        mine = {c: s.export_fd(c) for c in range(n_chunks) if own[c]}
        self._n_ranges += 1
        theirs = exchange_fds(self.rank, self.world, mine, self.group, tag=f"sap{self._n_ranges}")
        seen = set(mine)
        try:
            for sender, fds in theirs.items():
                for c, fd in fds.items():
                    if not 0 <= c < n_chunks or c in seen:
                        raise RuntimeError(f"rank {sender} sent chunk {c}, which is out of range or already mapped")
                    s.import_fd(c, fd)
                    seen.add(c)
        finally:
            for fds in theirs.values():
                for fd in fds.values():
                    os.close(fd)
            for fd in mine.values():
                os.close(fd)
        # a chunk nobody exported would stay an unmapped hole in the range: the kernels would fault on it much later
        missing = [c for c in range(n_chunks) if c not in seen]
        if missing:
            raise RuntimeError(f"rank {self.rank}: no process exported chunks {missing} of a {n_chunks}-chunk range")
        return s

    def tensor(self, tail_shape: Sequence[int], dtype):
        """[N, *tail_shape]: rows of chunk c are memory of the process that owns chunk c, mapped into this one."""
        import torch
        row = 1
        for x in tail_shape:
            row *= int(x)
        chunk_bytes = (self.n_tokens // self.P) * row * torch.empty((), dtype=dtype).element_size()
        s = self._assemble(self.P, chunk_bytes, [c in self.owned for c in range(self.P)])
        return s.tensor((self.n_tokens, *tail_shape), dtype, device=f"cuda:{self.device}")

    def own_rows(self) -> slice:
        n = self.n_tokens // self.P
        return slice(self.owned[0] * n, (self.owned[-1] + 1) * n)

    def shared(self, shape: Sequence[int], dtype):
        """One array for all ranks ([Hq, N] LSE, the backward workspace): memory of rank 0, mapped by every rank."""
        import torch
        nbytes = torch.empty((), dtype=dtype).element_size()
        for x in shape:
            nbytes *= int(x)
        g = api.Stitched.granularity(self.device)
        s = self._assemble(1, (nbytes + g - 1) // g * g, [self.rank == 0])
        return s.tensor(tuple(shape), dtype, device=f"cuda:{self.device}")

    def workspace(self, n_q_heads: int, n_kv_heads: int, head_dim: int):
        """The backward workspace; the accumulator rows of chunk c in the memory of the process that owns chunk c when the
        sizes line up (workspace_units), else one array in rank 0's memory."""
        import torch
        nbytes = api.sap_workspace_bytes(self.plan, n_q_heads, n_kv_heads, head_dim, api.SAP_PASS_BWD)
        lay = workspace_units(self.n_tokens, self.P, n_q_heads, head_dim, api.Stitched.granularity(self.device))
        if lay is None:
            return self.shared((nbytes,), torch.uint8)
        unit, per = lay
        own = [self.rank == 0] + [c in self.owned for c in range(self.P) for _ in range(per)]
        s = self._assemble(len(own), unit, own)
        return s.tensor((nbytes,), torch.uint8, device=f"cuda:{self.device}")

    def barrier(self):
        """Group barrier between phases: this rank's launches have finished and so have everybody else's."""
        import torch
        import torch.distributed as dist
        torch.cuda.synchronize()
        if self.world > 1:
            dist.barrier(group=self.group)

    @staticmethod
    def _ranges(chunks):
        """Chunks as [begin, end) runs: neighbours (7 and 8 of a zig-zag lap) share one launch."""
        runs, cs = [], sorted(chunks)
        for c in cs:
            if runs and runs[-1][1] == c:
                runs[-1][1] = c + 1
            else:
                runs.append([c, c + 1])
        return [(a, b) for a, b in runs]

    def forward(self, q, k, v, out, lse, softmax_scale: Optional[float] = None):
        for a, b in self._ranges(self.launch):
            api.sap_attn_fwd_chunks(q, k, v, self.cu_dev, self.plan, a, b, out, lse, softmax_scale=softmax_scale)

    def backward(self, dout, q, k, v, out, lse, dq, dk, dv, workspace, softmax_scale: Optional[float] = None):
        n_kv_heads = k.shape[1]
        self.barrier()         # every forward row (out, LSE) is written
        runs = self._ranges(self.launch)
        for a, b in runs:
            api.sap_attn_bwd_begin(dout, out, self.plan, a, b, n_kv_heads, workspace)
        self.barrier()         # every D written, every accumulator row zeroed
        for a, b in self._ranges(self.launch_kv):
            api.sap_attn_bwd_chunks(dout, q, k, v, lse, self.cu_dev, self.plan, a, b, dk, dv, workspace, softmax_scale=softmax_scale)
        self.barrier()         # every dQ contribution added
        for a, b in runs:
            api.sap_attn_bwd_end(self.plan, a, b, dq, n_kv_heads, workspace, softmax_scale=softmax_scale)
        self.barrier()
