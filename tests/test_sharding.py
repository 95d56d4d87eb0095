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


def _two_device_worker(rank, world, port, q):
    """One process per GPU: its own leb context on its own device, its slice of the batch, NCCL for the reductions."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import numpy as np
    from paper_2607_01203_b200 import leb, workloads as wl
    torch.cuda.set_device(rank)
    dev = torch.device("cuda", rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    w = wl.make_small_mlp([40, 64, 64, 64, 33], wl.ACT_TANH, 4, 6)       # wide enough for the tcgen05 path (200 KB smem launches)
    a, b = sharding.shard_range(w.B, rank, world)
    ctx = leb.context_for_workload(w, rank)
    lo, hi = ctx.leb_nn_fwd(torch.from_numpy(w.nom[a:b]).to(dev), torch.from_numpy(w.rad[a:b]).to(dev), flags=leb.FLAG_NO_MARGIN)
    torch.cuda.synchronize()
    n = sharding.sum_over_ranks(b - a, dev)
    q.put((rank, a, b, lo.cpu().numpy(), hi.cpu().numpy(), n))
    ctx.close()
    dist.destroy_process_group()


import pytest


@pytest.mark.gpu
def test_two_contexts_on_two_devices():
    """weights replicated, tiles partitioned, no collective on the data path.  Needs >= 2 GPUs (skipped on the
    1-GPU boxes this round has); also covers the per-device dynamic shared-memory attribute of the tcgen05 launches."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    from paper_2607_01203_b200 import build, leb, workloads as wl
    build.build()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_two_device_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=300) for _ in range(2)], key=lambda x: x[0])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    w = wl.make_small_mlp([40, 64, 64, 64, 33], wl.ACT_TANH, 4, 6)
    one = leb.context_for_workload(w, 0)
    lo, hi = one.leb_nn_fwd(torch.from_numpy(w.nom).cuda(), torch.from_numpy(w.rad).cuda(), flags=leb.FLAG_NO_MARGIN)
    got_lo = np.concatenate([r[3] for r in res]); got_hi = np.concatenate([r[4] for r in res])
    assert np.array_equal(got_lo, lo.cpu().numpy()) and np.array_equal(got_hi, hi.cpu().numpy())
    assert res[0][5] == w.B
    one.close()
