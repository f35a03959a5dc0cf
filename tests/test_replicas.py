"""N > 1 path of bench.py ("replicas only"): world_size-2 gloo test on CPU of the host logic."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1202_0635_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        seed = replicas.replica_seed(0x5EED0002, rank)
        # rank r pretends its K steps took 10 + 5 r ms and its end-to-end loop 100 - r ms
        mx = replicas.max_over_ranks([10.0 + 5.0 * rank, 100.0 - rank], dist)
        seeds = [None] * world
        dist.all_gather_object(seeds, seed)
        if rank == 0:
            out.put((mx, seeds, replicas.whole_job_ns_per_flip(mx[0], 4, 1 << 20, world)))
    finally:
        dist.destroy_process_group()


def test_two_replicas_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    mx, seeds, ns = out.get(timeout=120)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert mx == [15.0, 100.0]                      # slowest rank, per entry
    assert len(set(seeds)) == world and seeds[0] == 0x5EED0002
    assert ns == 15.0 * 1e6 / (2 * 4 * (1 << 20))   # all ranks' flips over the slowest rank's time


def test_single_process_passthrough():
    assert replicas.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert replicas.replica_seed(2 ** 64 - 1, 1) == 7918
