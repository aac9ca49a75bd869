"""Host-side logic of the N > 1 path on CPU: world_size 2 over gloo (DESIGN.md
"Multi-GPU": independent events per rank, no data-path collective; only the timing record
is reduced -- max of times, sum of units)."""
import os
import socket

import numpy as np
import pytest

import gen
from paper_2602_12052_b200 import shard


def test_shard_events_partition():
    for n in (0, 1, 2, 7, 10, 50):
        for world in (1, 2, 3, 8):
            got = [e for r in range(world) for e in shard.shard_events(n, world, r)]
            assert got == list(range(n))
            sizes = [len(shard.shard_events(n, world, r)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.shard_events(4, 2, 2)


def test_event_seeds_give_distinct_events():
    s0, s1 = shard.event_seed(1, 0), shard.event_seed(1, 1)
    assert s0 == 1001 and s1 != s0
    _, a = gen.make_segments(1, seed=s0)
    _, b = gen.make_segments(1, seed=s1)
    assert not np.array_equal(a["x0"], b["x0"])
    _, a2 = gen.make_segments(1, seed=s0)
    assert all(np.array_equal(a[k], a2[k]) for k in a)          # seeded: reproducible


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        events = list(shard.shard_events(5, world, rank))
        nseg = 0
        for e in events:
            _, segs = gen.make_segments(1, seed=shard.event_seed(1, e))
            nseg += len(segs["q"])
        ms, total = shard.reduce_timing([10.0 + rank, 3.0 - rank], nseg)
        q.put((rank, events, nseg, ms, total))
    finally:
        dist.destroy_process_group()


def test_world2_gloo_reduction():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, ev0, n0, ms0, tot0), (r1, ev1, n1, ms1, tot1) = res
    assert ev0 == [0, 1, 2] and ev1 == [3, 4]                   # no event on two ranks
    assert ms0 == ms1 == [11.0, 3.0]                            # max over ranks, per entry
    assert tot0 == tot1 == float(n0 + n1)                       # whole-job units


def test_reduce_timing_without_group():
    ms, n = shard.reduce_timing([1.5], 7)
    assert ms == [1.5] and n == 7.0
