"""World-size-2 gloo test (CPU) of the N > 1 host logic bench.py uses: barrier protocol, max over ranks, aggregate."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2309_06662_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        replicas.barrier(dist)
        ms_local = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
        ms = replicas.max_over_ranks(ms_local, dist)
        val = replicas.aggregate_throughput(1000, 4, ms, world)
        seeds = [None] * world
        dist.all_gather_object(seeds, replicas.replica_seed(6666, rank))
        replicas.barrier(dist)
        out.put((rank, ms, val, seeds))
    finally:
        dist.destroy_process_group()


def test_two_rank_protocol_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val, seeds in res:
        assert ms == 15.0                                 # max over ranks, identical on both
        assert val == 2 * 1000 * 4 / 15e-3                # whole-job aggregate
        assert seeds == [6666, 7666]                      # distinct ensemble members


def test_single_process_fallbacks():
    assert replicas.max_over_ranks(3.5, None) == 3.5
    assert replicas.aggregate_throughput(10, 2, 1.0, 1) == 20000.0
    replicas.barrier(None)
