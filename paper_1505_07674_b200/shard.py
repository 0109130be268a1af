"""Batch sharding over ranks: parameter vectors are independent and
the handle is read-only, so each rank holds a replica of the handle, evaluates a contiguous
slice of the batch and the only exchange is the all-gather of logL[B] (4 B bytes).  No
collective sits inside the path itself.
"""
import numpy as np


def shard_range(B, rank, world):
    """Contiguous slice [lo, hi) of a batch of B vectors for `rank` of `world`; sizes differ by
    at most one and the first B % world ranks get the longer slices."""
    if not (0 <= rank < world) or B < 0:
        raise ValueError("rank %d of %d, B = %d" % (rank, world, B))
    q, r = divmod(B, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def loglike_sharded(evaluate, params, rank=None, world=None, group=None):
    """logL[B] of the whole batch on every rank.

    evaluate(params_slice) -> tensor [n] float32 on the rank's device (on a GPU box: a closure
    around lensed.lensed_loglike); `params` is the full [B][P] tensor, identical on every rank.
    Uses torch.distributed (NCCL on GPUs, gloo in the CPU tests) for the one all-gather.
    """
    import torch
    import torch.distributed as dist
    if world is None:
        world = dist.get_world_size(group) if dist.is_initialized() else 1
        rank = dist.get_rank(group) if dist.is_initialized() else 0
    B = params.shape[0]
    lo, hi = shard_range(B, rank, world)
    mine = evaluate(params[lo:hi]) if hi > lo else torch.empty(0, dtype=torch.float32, device=params.device)
    if world == 1:
        return mine
    longest = shard_range(B, 0, world)
    pad = torch.full((longest[1] - longest[0],), float("nan"), dtype=torch.float32, device=mine.device)
    pad[: hi - lo] = mine
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    out = [parts[r][: np.subtract(*shard_range(B, r, world)[::-1])] for r in range(world)]
    return torch.cat(out)
