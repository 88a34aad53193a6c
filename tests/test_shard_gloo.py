"""The N > 1 path on CPU: world_size-2 gloo group.  Every rank takes its slice of the requests /
GPU ids, runs the per-unit computation (here the CPU oracle stands in for the device call — the
sharding logic is what is under test), gathers the records and must reproduce the unsharded result."""
from __future__ import annotations

import os
import socket
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import oracle
    from paper_2606_30391_b200 import shard, synth
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cl = synth.make_custom(seed=77, K=13, M=4, F=8, S=8, B=8, R=101, lo=1, hi=3)
    lo, hi = shard.shard_range(cl.R, rank, world)
    mine = oracle.place_batch(cl.lat, cl.pow, cl.models, cl.states, cl.requests[lo:hi])
    sizes = [shard.shard_range(cl.R, r, world)[1] - shard.shard_range(cl.R, r, world)[0] for r in range(world)]
    full = shard.gather_records(mine, sizes, dist)
    glo, ghi = shard.shard_range(cl.K, rank, world)
    lmine = oracle.local_config(cl.lat, cl.pow, cl.states, 0, np.arange(glo, ghi, dtype=np.int32))
    lsizes = [shard.shard_range(cl.K, r, world)[1] - shard.shard_range(cl.K, r, world)[0] for r in range(world)]
    lfull = shard.gather_records(lmine, lsizes, dist)
    # the same exchange from a torch byte tensor (what a FS_DEVICE call leaves behind), with the record dtype
    import torch
    tfull = shard.gather_records(torch.from_numpy(mine.view(np.uint8).reshape(-1).copy()), sizes, dist, dtype=mine.dtype)
    assert tfull.tobytes() == full.tobytes()
    if rank == 0:
        ref = oracle.place_batch(cl.lat, cl.pow, cl.models, cl.states, cl.requests)
        lref = oracle.local_config(cl.lat, cl.pow, cl.states, 0)
        ok = full.tobytes() == ref.tobytes() and lfull.tobytes() == lref.tobytes()
        open(os.path.join(out_dir, "ok"), "w").write("1" if ok else "0")
    dist.barrier()
    dist.destroy_process_group()


def test_shard_range_partitions():
    from paper_2606_30391_b200 import shard
    for n in (0, 1, 7, 64, 65536):
        for w in (1, 2, 3, 8):
            spans = [shard.shard_range(n, r, w) for r in range(w)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.shard_range(4, 2, 2)


def test_two_rank_gloo_gather_equals_unsharded(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    assert open(tmp_path / "ok").read() == "1"
