"""The N>1 plumbing of the batch path on CPU: world_size-2 gloo processes."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1507_08549_b200.sharding import reduce_timing, shard_members


def test_shards_partition_the_batch():
    for n in (2, 3, 64, 65):
        for world in (1, 2, 4, 8):
            if n < world:
                continue
            seen = []
            for r in range(world):
                idx, mode = shard_members(n, r, world)
                assert mode == "strong"
                seen += idx
            assert sorted(seen) == list(range(n))
            sizes = [len(shard_members(n, r, world)[0]) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


def test_single_solve_runs_as_replicas():
    for world in (1, 2, 8):
        for r in range(world):
            assert shard_members(1, r, world) == ([0], "weak")
    assert shard_members(3, 1, 4) == ([0, 1, 2], "weak")
    with pytest.raises(ValueError):
        shard_members(4, 2, 2)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        idx, mode = shard_members(7, rank, world)
        # a rank's "device time" and work counters, as bench.py feeds them
        ms = 10.0 + 5.0 * rank
        upd = float(sum(100 + i for i in idx))
        dist.barrier()
        tmax, (usum, lsum) = reduce_timing(ms, [upd, float(len(idx))], world)
        q.put((rank, idx, mode, tmax, usum, lsum))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_reduction():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, i0, m0, t0, u0, l0), (r1, i1, m1, t1, u1, l1) = out
    assert m0 == m1 == "strong"
    assert sorted(i0 + i1) == list(range(7)) and not set(i0) & set(i1)
    assert t0 == t1 == 15.0                                   # max over ranks
    assert u0 == u1 == float(sum(100 + i for i in range(7)))  # whole-job work
    assert l0 == l1 == 7.0


def test_world_size_1_needs_no_process_group():
    assert reduce_timing(3.5, [1, 2], 1) == (3.5, [1.0, 2.0])
