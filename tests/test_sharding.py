"""Multi-GPU path: tiles are independent, so ranks take contiguous slices of the
batch and no collective is on the data path.  The partition logic is exercised here with
world_size-2 gloo processes on CPU (no kernels are launched)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_01203_b200 import sharding


def test_shard_ranges_cover_exactly_once():
    for total in (0, 1, 7, 64, 6400):
        for world in (1, 2, 3, 8):
            spans = [sharding.shard_range(total, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == total
            for (a, b), (c, d) in zip(spans, spans[1:]):
                assert b == c and a <= b
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, total, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    a, b = sharding.shard_range(total, rank, world)
    # each rank "processes" its slice (stand-in for the kernels): marks the tiles it owns
    owned = torch.zeros(total, dtype=torch.int32)
    owned[a:b] = 1
    # timing is max over ranks; the count of processed units is summed (bench.py's reduction)
    t = sharding.max_over_ranks(float(rank + 1))
    n = sharding.sum_over_ranks(b - a)
    gathered = [torch.zeros(total, dtype=torch.int32) for _ in range(world)]
    dist.all_gather(gathered, owned)
    if rank == 0:
        out.put((t, n, torch.stack(gathered).sum(0).numpy()))
    dist.destroy_process_group()


def test_world_size_2_gloo_partition_and_reductions():
    world, total = 2, 101
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, total, q)) for r in range(world)]
    for p in procs:
        p.start()
    t, n, cover = q.get(timeout=120)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert t == 2.0 and n == total
    assert np.all(cover == 1)
