"""Multi-GPU plumbing: theta vectors are independent, so the batch is sharded across ranks
with no data-path collective; grid, PSF, data, errors and mask (<= 1.5 MB) are replicated.  The only exchanges are
the max-over-ranks of the device time and the gather of logL, both through torch.distributed (NCCL on GPUs,
gloo in the CPU tests).  Nothing here computes any part of the model."""
from __future__ import annotations

import os

import numpy as np


def env_rank_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))


def shard_bounds(B: int, rank: int, world: int):
    """Contiguous, balanced [lo, hi) of rank's shard of a batch of B (the first B % world ranks get one more)."""
    base, rem = divmod(B, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def shard(theta: np.ndarray, rank: int, world: int) -> np.ndarray:
    lo, hi = shard_bounds(theta.shape[0], rank, world)
    return theta[lo:hi]


def _reduce_device(device):
    """Where a scalar to be all-reduced must live: NCCL reduces CUDA tensors only, gloo takes CPU tensors."""
    import torch.distributed as dist
    if device is not None:
        return device
    return "cuda" if dist.get_backend() == "nccl" else "cpu"


def max_over_ranks(value: float, device=None) -> float:
    """max of a per-rank scalar (device time); identity when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=_reduce_device(device))
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=_reduce_device(device))
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_logl(local, B: int, rank: int, world: int):
    """All-gather the per-rank logL shards (torch tensors) into the full [B] vector, in batch order."""
    import torch
    import torch.distributed as dist
    if world == 1 or not (dist.is_available() and dist.is_initialized()):
        return local
    sizes = [shard_bounds(B, r, world)[1] - shard_bounds(B, r, world)[0] for r in range(world)]
    pad = max(sizes)
    buf = torch.zeros(pad, dtype=local.dtype, device=local.device)
    buf[: local.numel()] = local
    out = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(out, buf)
    return torch.cat([o[:n] for o, n in zip(out, sizes)])


def loglike_sharded(ctx, theta, rank: int | None = None, world: int | None = None):
    """SURVEY.md sec. 8(e) as one call: theta[B][17] (the same full batch on every rank) -> logL[B] on every rank.
    Each rank evaluates its contiguous shard with `ctx.loglike` (any object with that method: a bang.Context bound
    to the rank's GPU) and the shards are all-gathered in batch order.  No collective touches the data path."""
    import torch
    import torch.distributed as dist
    if rank is None or world is None:
        on = dist.is_available() and dist.is_initialized()
        rank, world = (dist.get_rank(), dist.get_world_size()) if on else (0, 1)
    B = theta.shape[0]
    lo, hi = shard_bounds(B, rank, world)
    local = ctx.loglike(theta[lo:hi]) if hi > lo else torch.empty(0, dtype=torch.float64, device=getattr(ctx, "device", "cpu"))
    return gather_logl(local, B, rank, world)
