"""world_size-2 gloo test (CPU) of the multi-GPU host logic: time-step sharding with no collective
on the data path, and the barrier + max-over-ranks timing reduction bench.py uses."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2405_13478_b200 import shard, synth


def test_shard_partition_properties():
    for n_t in (0, 1, 5, 100, 101):
        for world in (1, 2, 3, 8):
            parts = [shard.shard_time_steps(n_t, world, r) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n_t
            assert all(parts[r][1] == parts[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in parts]
            assert max(sizes) - min(sizes) <= 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = synth.config_station(n_t=5, n_ch=2, n_pix=32)
        t0, t1 = shard.shard_time_steps(w.n_t, world, rank)
        vis = w.vis(t0, t1)                                   # each rank generates only its shard
        full = w.vis()
        assert np.array_equal(vis, full[t0:t1])               # shards are slices of the same batch
        dist.barrier()
        units = (t1 - t0) * w.n_ch
        thr, ms = shard.aggregate_throughput(units, 10.0 * (rank + 1))
        assert ms == 10.0 * world                             # MAX over ranks
        assert abs(thr - w.n_t * w.n_ch / (ms / 1e3)) < 1e-9   # all units / slowest rank's time
        out.put((rank, t0, t1))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_sharding_and_timing():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    got = sorted(out.get(timeout=10) for _ in range(world))
    assert got == [(0, 0, 3), (1, 3, 5)]
