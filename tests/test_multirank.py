"""-m "not gpu": the N > 1 path of bench.py (independent problems per rank, max-over-ranks timing) with
world_size-2 gloo on CPU.  No data-path collective exists."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import emugemm_inputs as G
from paper_2606_25453_b200 import shard


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seed = shard.rank_seed(1, rank)
    A, _ = G.real_pair(8, 8, 8, 0.5, seed)
    ms = shard.max_over_ranks(10.0 + 5.0 * rank, dist)  # rank 1 is the slow one
    # every rank sees the same max; the problems differ
    gathered = [None] * world
    dist.all_gather_object(gathered, (seed, float(A[0, 0]), ms))
    if rank == 0:
        out.put(gathered)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_independent_problems_and_max_timing():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (s0, a0, ms0), (s1, a1, ms1) = res
    assert (s0, s1) == (1, 1001) and a0 != a1
    assert ms0 == ms1 == 15.0
    assert shard.aggregate_throughput(2.0, 2, 15.0) == 2 * 2.0 / 0.015


def test_single_process_identity():
    assert shard.max_over_ranks(3.5) == 3.5
    assert shard.rank_seed(4, 0) == 4
