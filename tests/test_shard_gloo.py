"""The N > 1 bookkeeping on CPU: plane ranges and max-over-ranks with gloo, world size 2."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1503_07998_b200 import shard


@pytest.mark.parametrize("n,world", [(512, 2), (511, 2), (7, 4), (1, 2), (0, 3), (2048, 8), (10, 3)])
def test_plane_ranges_partition_the_stack_on_even_boundaries(n, world):
    r = [shard.plane_range(n, k, world) for k in range(world)]
    assert r[0][0] == 0 and r[-1][1] == n
    for (a0, a1), (b0, b1) in zip(r, r[1:]):
        assert a1 == b0 and a0 <= a1
    assert all(p0 % 2 == 0 for p0, _ in r)
    sizes = [p1 - p0 for p0, p1 in r]
    assert max(sizes) - min(sizes) <= 3          # one pair, plus the odd tail


def test_plane_range_rejects_bad_arguments():
    with pytest.raises(ValueError):
        shard.plane_range(8, 2, 2)
    with pytest.raises(ValueError):
        shard.plane_range(-1, 0, 1)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_planes, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        p0, p1 = shard.plane_range(n_planes, rank, world)
        # every rank "processes" its planes; rank r pretends to take (r + 1) * 10 ms
        t = shard.max_over_ranks(0.010 * (rank + 1))
        counts = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(counts, torch.tensor([p1 - p0]))
        dist.barrier()
        q.put((rank, p0, p1, t, [int(c) for c in counts]))
    finally:
        dist.destroy_process_group()


def test_two_ranks_agree_on_the_slowest_time_and_cover_all_planes():
    world, n = 2, 511
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[3] for g in got] == [pytest.approx(0.020)] * 2       # MAX over ranks, same on both
    assert got[0][1] == 0 and got[0][2] == got[1][1] and got[1][2] == n
    assert got[0][4] == got[1][4] and sum(got[0][4]) == n
    assert shard.job_throughput([u * 100 for u in got[0][4]], got[0][3]) == pytest.approx(n * 100 / 0.020)


def test_max_over_ranks_is_identity_without_a_group():
    assert shard.max_over_ranks(1.25) == 1.25
    assert shard.job_throughput(10, 2.0, world=4) == 20.0
