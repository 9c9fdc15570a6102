"""Multi-GPU plumbing: photons are independent (paper P:39), so a batch is split into contiguous photon
ranges, one per rank, and integrated with no exchange.  The only data that ever crosses ranks is the result:
status bytes of an image (to assemble the capture map on one rank) and a few counters.  torch.distributed only;
nothing here touches the photon states and there is no arithmetic of the method in this module.
"""
import torch
import torch.distributed as dist

from .workloads import shard_range


def gather_bytes(local, n_total, group=None):
    """All ranks hold `local`, the uint8 slice [lo, hi) = shard_range(n_total, rank, world) of an n_total-byte
    array (e.g. the `status` of their photons); returns the whole array on every rank.  Slices may be uneven:
    they are padded to the largest one for the collective and trimmed afterwards."""
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    lo, hi = shard_range(n_total, rank, world)
    if local.dtype != torch.uint8 or local.numel() != hi - lo:
        raise ValueError(f"rank {rank}: expected {hi - lo} bytes, got {local.numel()} of {local.dtype}")
    width = max(shard_range(n_total, r, world)[1] - shard_range(n_total, r, world)[0] for r in range(world))
    padded = torch.zeros((width,), dtype=torch.uint8, device=local.device)
    padded[: hi - lo] = local
    parts = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(parts, padded, group=group)
    out = torch.empty((n_total,), dtype=torch.uint8, device=local.device)
    for r in range(world):
        a, b = shard_range(n_total, r, world)
        out[a:b] = parts[r][: b - a]
    return out


def sum_counters(counters, device, group=None):
    """Element-wise sum over ranks of a dict of integer counters (gray_integrate_counters, status histogram)."""
    keys = sorted(counters)
    t = torch.tensor([int(counters[k]) for k in keys], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return {k: int(v) for k, v in zip(keys, t.tolist())}


def max_time_ms(ms, device, group=None):
    """Device time of a multi-GPU step = max over ranks."""
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
