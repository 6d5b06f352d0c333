"""World-size-2 gloo test (CPU) of the multi-GPU host logic of bench.py: the path does not
shard within a solve (replicas only), so the N > 1 logic is the
assignment of disjoint sources to ranks and the max/sum reduction of the timing scalars."""
import os
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ids = bench.rank_sources(rank, 12)
        secs, (iters, launches) = bench.reduce_over_ranks(1.0 + rank, [100 * (rank + 1), 7], None)
        q.put((rank, ids, secs, iters, launches))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, ids0, s0, it0, l0), (r1, ids1, s1, it1, l1) = res
    assert ids0 == list(range(0, 12)) and ids1 == list(range(12, 24))  # disjoint, contiguous
    assert s0 == s1 == 2.0            # max over ranks
    assert it0 == it1 == 300          # sum over ranks
    assert l0 == l1 == 14


def test_single_process_identity():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.reduce_over_ranks(1.5, [3, 4]) == (1.5, [3, 4])
    assert bench.rank_sources(0, 4) == [0, 1, 2, 3]
