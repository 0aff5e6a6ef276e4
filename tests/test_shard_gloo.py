"""N > 1 path on CPU: the sharding helper and the two scalar reductions of bench.py / a multi-GPU driver, run with
world_size 2 over gloo (the path has no data collective)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1804_03479_b200 import shard


def test_shard_range_partitions_exactly():
    for G in (0, 1, 7, 512, 513):
        for world in (1, 2, 3, 8):
            parts = [shard.shard_range(G, r, world) for r in range(world)]
            assert sum(c for _, c in parts) == G
            assert parts[0][0] == 0
            for (f0, c0), (f1, _) in zip(parts, parts[1:]):
                assert f0 + c0 == f1
            assert max(c for _, c in parts) - min(c for _, c in parts) <= 1
    with pytest.raises(ValueError):
        shard.shard_range(4, 2, 2)


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # every rank owns a shard of 513 groups and a local max signal speed / device time
        first, count = shard.shard_range(513, rank, world)
        local_speed = 1.0 + 0.5 * rank
        local_ms = 10.0 - 3.0 * rank
        dt = shard.global_dt(local_speed, dh=1.0 / 16, cfl=0.3, dist=dist)
        ms = shard.max_over_ranks(local_ms, dist)
        total = torch.tensor([float(count)], dtype=torch.float64)
        dist.all_reduce(total)
        out.put((rank, first, count, dt, ms, float(total.item())))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_reductions():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, f0, c0, dt0, ms0, t0), (r1, f1, c1, dt1, ms1, t1) = res
    assert (f0, c0, f1, c1) == (0, 257, 257, 256) and t0 == t1 == 513.0
    assert dt0 == dt1 == 0.3 * (1.0 / 16) / 1.5          # the slowest rank's signal speed sets the global dt
    assert ms0 == ms1 == 10.0                              # the slowest rank's device time is the job's time
