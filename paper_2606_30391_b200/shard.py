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


def gather_records(local, world_sizes, dist, group=None, dtype=None):
    """All-gather variable-length record arrays (as bytes) over torch.distributed and concatenate them in
    rank order.  `world_sizes[r]` = number of records of rank r.
    `local` is a numpy record array (host) or a torch uint8 tensor holding records of numpy `dtype` (host or
    CUDA: the device buffer a FS_DEVICE call wrote).  The exchange runs where the group's backend needs it: CUDA
    tensors on an NCCL group (ncclAllGather over NVLink; host arrays are staged to the current device), host
    tensors on gloo.  Returns a numpy record array on every rank."""
    import numpy as np
    import torch
    if isinstance(local, torch.Tensor):
        if dtype is None:
            raise ValueError("dtype is required with a tensor")
        dtype = np.dtype(dtype)
        raw = local.reshape(-1).view(torch.uint8)
    else:
        dtype = local.dtype
        raw = torch.from_numpy(np.ascontiguousarray(local).view(np.uint8).reshape(-1).copy())
    item = dtype.itemsize
    nccl = dist.get_backend(group) == "nccl"
    dev = torch.device("cuda", torch.cuda.current_device()) if nccl else torch.device("cpu")
    cap = max(max(world_sizes) * item, 1)
    buf = torch.zeros(cap, dtype=torch.uint8, device=dev)
    buf[: raw.numel()] = raw.to(dev)
    outs = [torch.zeros_like(buf) for _ in world_sizes]
    dist.all_gather(outs, buf, group=group)
    parts = [o.cpu().numpy()[: n * item].view(dtype) for o, n in zip(outs, world_sizes)]
    return np.concatenate(parts) if parts else np.zeros(0, dtype=dtype)
