"""world_size-2 gloo test (CPU) of the N>1 host logic: contiguous sharding of a batch and the all-gather of the
per-rank log-likelihoods.  The GPU kernels themselves have no cross-rank dependency."""
import os
import socket

import numpy as np
import torch
import torch.multiprocessing as mp

from paper_2504_01302_b200.sharding import gather_loglike, shard_range


def test_shard_ranges_tile_the_batch():
    for B in (0, 1, 7, 8, 1024, 1025):
        for world in (1, 2, 3, 8):
            spans = [shard_range(B, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == B
            assert all(spans[i][1] == spans[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, B, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    full = torch.arange(B, dtype=torch.float32) * -0.5 - 3.0          # stands for the lnL of vector b
    lo, hi = shard_range(B, rank, world)
    got = gather_loglike(full[lo:hi].clone(), B, rank, world, dist)
    q.put((rank, bool(torch.equal(got, full))))
    dist.destroy_process_group()


def test_two_rank_gather_of_ragged_batch():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, 1025, q)) for r in range(2)]
    [p.start() for p in procs]
    res = sorted(q.get(timeout=120) for _ in procs)
    [p.join(timeout=60) for p in procs]
    assert res == [(0, True), (1, True)]
