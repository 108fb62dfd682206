"""The N > 1 path on CPU: theta sharding, max-over-ranks timing and the logL gather, world_size 2 over gloo."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_bounds_partition_the_batch():
    from paper_2205_06819_b200 import dist as D
    for B in (0, 1, 7, 1024, 16385):
        for world in (1, 2, 3, 8):
            edges = [D.shard_bounds(B, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == B
            assert all(edges[i][1] == edges[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in edges]
            assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, B, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2205_06819_b200 import dist as D
    from paper_2205_06819_b200 import workloads as W
    theta = W.theta_batch(2, B)
    mine = D.shard(theta, rank, world)
    # stand-in for the per-rank likelihood: any function of the rank's own theta rows (the real one needs a GPU)
    local = torch.as_tensor(mine.sum(axis=1))
    full = D.gather_logl(local, B, rank, world)

    class StubContext:                       # the same stand-in behind bang.Context's loglike(theta) -> logL interface
        device = "cpu"

        def loglike(self, th):
            return torch.as_tensor(np.asarray(th).sum(axis=1))

    sharded = D.loglike_sharded(StubContext(), theta)          # the sec. 8(e) entry point: shard -> evaluate -> all-gather
    assert torch.equal(sharded, full)
    t = D.max_over_ranks(1.0 + rank)
    n = D.sum_over_ranks(float(len(mine)))
    q.put((rank, full.numpy(), t, n))
    dist.destroy_process_group()


@pytest.mark.parametrize("B", [10, 1023])
def test_world_size_two_gloo(B):
    from paper_2205_06819_b200 import workloads as W
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() + B) % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, B, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    want = W.theta_batch(2, B).sum(axis=1)
    for rank, full, t, n in res:
        assert np.array_equal(full, want)        # every rank ends with the whole batch, in order
        assert t == 2.0 and n == B               # max over ranks of the time; shards cover the batch
