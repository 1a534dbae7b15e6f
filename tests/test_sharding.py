"""N > 1 host logic on CPU: disjoint quartet ranges per rank and the max-over-ranks timing reduction
(world size 2, gloo backend, 127.0.0.1)."""
import os
import socket

import numpy as np
import pytest

from paper_2405_01834_b200 import sharding, workloads as W


@pytest.mark.parametrize("n,world", [(0, 1), (1, 2), (7, 2), (200000, 8), (5, 8), (13, 4)])
def test_shard_range_partitions(n, world):
    got = [sharding.shard_range(n, r, world) for r in range(world)]
    assert got[0][0] == 0 and got[-1][1] == n
    assert all(a[1] == b[0] for a, b in zip(got, got[1:]))
    sizes = [hi - lo for lo, hi in got]
    assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = W.config1(64)                                   # every rank sees the same seeded workload
        lo, hi = sharding.shard_range(w.nquartets, rank, world)
        ia, _, _, _ = w.shell_indices(np.arange(lo, hi))
        t = sharding.max_over_ranks(1.0 + rank)             # "time" of this rank
        q.put((rank, lo, hi, int(ia.sum()), t))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_shards_and_max_time():
    import torch.multiprocessing as mp
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, lo0, hi0, s0, t0), (r1, lo1, hi1, s1, t1) = res
    assert (lo0, hi0, lo1, hi1) == (0, 32, 32, 64)
    assert s0 + s1 == sum(range(64))                        # disjoint cover of the quartet list
    assert t0 == t1 == 2.0                                  # MAX over ranks, seen by both
