"""CPU, world_size 2, gloo: the host-side logic of bench.py's N > 1 path (source sharding, max-over-ranks timing).
The oracle's noise stands in for the device noise (same spec): shards of different ranks must tile the global stream."""
import os
import socket

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1405_4524_b200 import sharding


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    dims, n = (2, 2, 2, 4), 3
    off = sharding.source_offset(rank, n)
    mine = oracle.noise_fill(dims, 77, n, rhs_offset=off, scale=1.0)
    ms = sharding.max_over_ranks(10.0 + 5.0 * rank)           # rank 1 is slower
    q.put((rank, off, mine.tobytes(), ms))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_tile_the_source_stream_and_reduce_time():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    import oracle
    full = oracle.noise_fill((2, 2, 2, 4), 77, 6, scale=1.0)
    assert [g[1] for g in got] == [0, 3]
    assert got[0][2] + got[1][2] == full.tobytes()            # shards tile the global stream, no overlap
    assert all(g[3] == 15.0 for g in got)                     # max over ranks
    assert sharding.whole_job_seconds_per_source(15.0, 3, 3, 2) == 15e-3 / 18


def test_source_slices():
    assert sharding.source_slices(32, 4) == [(0, 8), (8, 8), (16, 8), (24, 8)]
    assert sharding.source_slices(7, 3) == [(0, 3), (3, 2), (5, 2)]
    assert sum(c for _, c in sharding.source_slices(64, 8)) == 64
