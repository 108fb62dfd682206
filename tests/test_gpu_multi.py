"""Two GPUs: each rank's context lives on ITS device, `dist.loglike_sharded` (SURVEY.md sec. 8e as one call)
returns on every rank the vector the single-GPU call returns, and creating a context on another device leaves the calling
thread's current device alone.  Skipped where fewer than two CUDA devices are visible (the GPU pool of this build has one
per box); the host side of the same function is covered on CPU by tests/test_dist_gloo.py."""
import os

import numpy as np
import pytest

from paper_2205_06819_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _rank(rank, world, port, q):
    import torch
    import torch.distributed as dist
    from paper_2205_06819_b200 import bang, dist as D
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    cfg = W.config(2)
    c64 = bang.Context(cfg, precision="fp64", device=rank)
    mtrue = c64.model_maps(W.theta_true(2)).cpu().numpy()[0]
    c64.close()
    data, err, mask = W.make_data(2, mtrue)
    ctx = bang.Context(cfg, precision="fp32", device=rank)
    ctx.set_data(data, err, mask)
    assert ctx.device == torch.device("cuda", rank) and torch.cuda.current_device() == rank
    theta = torch.as_tensor(W.theta_batch(2)[:301], device=ctx.device)       # 301: ragged shards
    full = D.loglike_sharded(ctx, theta)
    assert full.device == ctx.device and full.shape == (301,)
    single = ctx.loglike(theta)
    ok = bool(torch.equal(full, single))
    other = bang.Context(cfg, precision="fp32", device=(rank + 1) % world)   # a context on the OTHER device ...
    still = torch.cuda.current_device() == rank                               # ... does not move this thread's device
    other.close()
    ctx.close()
    q.put((rank, ok, still, full.cpu().numpy()))
    dist.destroy_process_group()


def test_two_gpus_shard_and_gather():
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_rank, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=300) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(ok and still for _, ok, still, _ in res)
    assert np.array_equal(res[0][3], res[1][3])
