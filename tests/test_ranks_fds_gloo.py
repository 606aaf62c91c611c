"""ranks.exchange_fds on CPU: three gloo ranks hand each other file descriptors over Unix sockets (SCM_RIGHTS) - the
transport the one-process-per-GPU form of the stitched allocation uses for its exported chunks.  Here the descriptors
are unlinked temporary files: what a rank writes into its own file must be readable through the descriptor its peers
received (same open file, no path involved)."""
import os
import socket
import tempfile

import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2606_30460_b200.ranks import exchange_fds
        files = {key: tempfile.TemporaryFile() for key in (10 * rank, 10 * rank + 1)} if rank != 2 else {}   # rank 2 owns nothing
        got = exchange_fds(rank, world, {k: f.fileno() for k, f in files.items()})
        for k, f in files.items():
            os.pwrite(f.fileno(), f"from {rank} key {k}".encode(), 0)
        dist.barrier()
        seen = {}
        for sender, fds in got.items():
            for k, fd in fds.items():
                seen[(sender, k)] = os.pread(fd, 64, 0).decode()
                os.close(fd)
        q.put((rank, seen))
    finally:
        dist.destroy_process_group()


def test_three_ranks_exchange_descriptors():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 3, port, q)) for r in range(3)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    want = {(s, k): f"from {s} key {k}" for s in (0, 1) for k in (10 * s, 10 * s + 1)}
    for rank in range(3):
        assert res[rank] == {sk: v for sk, v in want.items() if sk[0] != rank}, (rank, res[rank])


def _bad_peer_worker(rank, world, port, q):
    """rank 1 speaks the protocol by hand and announces two keys while attaching one descriptor; rank 0 must refuse"""
    import array
    import struct
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        if rank == 0:
            from paper_2606_30460_b200.ranks import exchange_fds
            try:
                exchange_fds(0, 2, {})
                q.put("accepted")
            except RuntimeError as e:
                q.put(str(e))
        else:
            box = [None]
            dist.broadcast_object_list(box, src=0)
            assert oct(os.stat(box[0]).st_mode & 0o777) == "0o700"      # private to this user
            srv = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)     # rank 0 sends its (empty) message here
            srv.bind(os.path.join(box[0], "1"))
            srv.listen(2)
            dist.barrier()
            with tempfile.TemporaryFile() as f:
                c = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)
                c.connect(os.path.join(box[0], "0"))
                c.sendmsg([struct.pack("<iiii", 1, 2, 7, 8)], [(socket.SOL_SOCKET, socket.SCM_RIGHTS, array.array("i", [f.fileno()]))])
                c.close()
    finally:
        dist.destroy_process_group()


def test_incomplete_message_is_refused():
    from paper_2606_30460_b200.ranks import exchange_fds
    import pytest
    with pytest.raises(ValueError):          # more descriptors than one SCM_RIGHTS message carries: refused before anything is sent
        exchange_fds(0, 2, {i: 0 for i in range(254)})
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_bad_peer_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    msg = q.get(timeout=120)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert "malformed or foreign message" in msg and "2 keys" in msg and "1 descriptors" in msg, msg


def test_launch_chunks_cover_every_chunk_once_and_balance_the_causal_load():
    """ranks.launch_chunks: a partition of the chunks; with one document over the whole sequence the work of q-chunk c
    is c + 1 blocks, and zig-zag brings every rank to the same total where contiguous ownership does not."""
    from paper_2606_30460_b200.ranks import launch_chunks
    for world, P in ((2, 4), (4, 16), (8, 16), (3, 9), (2, 2)):
        for balance in ("zigzag", "contiguous"):
            L = [launch_chunks(r, world, P, balance) for r in range(world)]
            assert sorted(sum(L, [])) == list(range(P))
        zz = [sum(c + 1 for c in launch_chunks(r, world, P)) for r in range(world)]
        ct = [sum(c + 1 for c in launch_chunks(r, world, P, "contiguous")) for r in range(world)]
        if (P // world) % 2 == 0:
            assert max(zz) == min(zz) and max(ct) > min(ct)
        assert max(zz) <= max(ct)


def test_work_balanced_assignment():
    """ranks.chunk_work / assign_by_work: the per-chunk work sums to the useful pairs of the sequence (both ways of
    counting), the assignment is a partition, and greedy LPT is within one chunk's work of the mean."""
    from paper_2606_30460_b200.ranks import assign_by_work, chunk_work
    from paper_2606_30460_b200.workloads import make_workload
    for cfg in (1, 2, 3, 4, 5):
        w = make_workload(cfg)
        q_work, kv_work = chunk_work(w.cu_seqlens, w.n_chunks)
        assert sum(q_work) == w.pairs == sum(kv_work)
        for world in (1, 2, 4):
            for work in (q_work, kv_work):
                a = assign_by_work(work, world)
                assert sorted(sum(a, [])) == list(range(w.n_chunks))
                loads = [sum(work[c] for c in x) for x in a]
                assert max(loads) - min(loads) <= max(work)
    # one document: q-chunk c costs about (2c + 1) blocks; LPT pairs cheap with expensive chunks like zig-zag does
    q_work, _ = chunk_work([0, 8192], 8)
    loads = [sum(q_work[c] for c in x) for x in assign_by_work(q_work, 4)]
    assert max(loads) / (sum(loads) / 4) < 1.01
