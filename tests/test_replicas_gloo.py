"""world_size-2 gloo test of the multi-GPU host logic (replicas only: per-rank seeds, max-over-ranks timing,
whole-job throughput). Runs on CPU."""
import os

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2306_04322_b200 import replicas, synth


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        per_rank = 3
        seeds = [replicas.replica_seed(7, rank, r, per_rank) for r in range(per_rank)]
        c, _ = synth.init_a((16, 16), 1, seeds[0])
        c = replicas.perturb(c, rank, 0, per_rank)
        elapsed = 10.0 + 5.0 * rank                              # rank 1 is the slow one
        tmax = replicas.max_over_ranks(elapsed)
        value = replicas.job_throughput(100, tmax, world)
        gathered = [None] * world
        dist.all_gather_object(gathered, (seeds, float(c.mean())))
        if rank == 0:
            out.put((tmax, value, gathered))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_rank_replica_logic():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    tmax, value, gathered = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert tmax == 15.0                                           # max over ranks, not rank 0's own time
    assert np.isclose(value, 2 * 100 / 15e-3)
    all_seeds = gathered[0][0] + gathered[1][0]
    assert len(set(all_seeds)) == 6                               # no two replicas share a seed
    assert gathered[0][1] != gathered[1][1]


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.job_throughput(10, 1000.0, 1) == 10.0
