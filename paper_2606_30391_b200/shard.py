"""Host-side partition of the hot path over ranks (one process per GPU).

The path has no exchange step: requests (fs_place_batch), GPU ids (fs_local_config) and sources
(fs_consolidate) are independent units, so N ranks each take a contiguous, balanced slice with
tables and state replicated.  Results are gathered by the caller (32/48/16-byte records)."""
from __future__ import annotations


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """[lo, hi) of rank's slice of n units: sizes differ by at most one, order preserved."""
    if not (0 <= rank < world) or n < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def gather_records(local, world_sizes, dist, group=None):
    """All-gather variable-length numpy record arrays (as bytes) over torch.distributed and
    concatenate them in rank order.  `world_sizes[r]` = number of records of rank r."""
    import numpy as np
    import torch
    item = local.dtype.itemsize
    cap = max(world_sizes) * item
    buf = torch.zeros(max(cap, 1), dtype=torch.uint8)
    raw = np.ascontiguousarray(local).view(np.uint8).reshape(-1)
    buf[: raw.size] = torch.from_numpy(raw.copy())
    outs = [torch.zeros_like(buf) for _ in world_sizes]
    dist.all_gather(outs, buf, group=group)
    parts = [o.numpy()[: n * item].view(local.dtype) for o, n in zip(outs, world_sizes)]
    return np.concatenate(parts) if parts else local[:0]
