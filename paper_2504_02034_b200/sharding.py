"""Multi-GPU host logic: the path shards by lambda with no data-path collective.

Every (event, lambda) and (injection, lambda) evaluation is independent, so rank r of W takes a contiguous
slice of the lambda batch, inputs are replicated, and the only exchange is the final gather of n_lambda
doubles (torch.distributed all_gather; NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations


def shard_lambda(n_lambda: int, rank: int, world: int):
    """Contiguous, balanced slice [lo, hi) of the lambda batch owned by `rank` (sizes differ by at most 1)."""
    if world < 1 or not (0 <= rank < world) or n_lambda < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(n_lambda, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def gather_lambda_results(local, n_lambda: int, group=None):
    """all_gather the per-rank result slices (1-D tensors, possibly of unequal length) into one [n_lambda] tensor."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    sizes = [shard_lambda(n_lambda, r, world) for r in range(world)]
    width = max(hi - lo for lo, hi in sizes)
    pad = torch.zeros(width, dtype=local.dtype, device=local.device)
    pad[: local.numel()] = local
    bufs = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(bufs, pad, group=group)
    return torch.cat([b[: hi - lo] for b, (lo, hi) in zip(bufs, sizes)])
