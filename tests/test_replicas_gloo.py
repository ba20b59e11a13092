"""N > 1 host logic (replicas only) on CPU: world_size 2, gloo backend, rendezvous on 127.0.0.1.
Checks the per-rank seeding (ranks simulate different instances), the barrier and the max-over-ranks reduction
bench.py uses, and that nothing on this path needs a collective on simulation data."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2405_14903_b200 import replicas, workloads as wl


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        r, w, _ = replicas.rank_world()
        assert (r, w) == (rank, world)
        P = wl.config4_params(16, seed=1004 + replicas.seed_shift(r))
        U0 = wl.config4_initial_velocity(P)
        checksum = float(np.sum(U0[0].astype(np.float64)))
        replicas.barrier(dist)
        local_ms = 10.0 + 5.0 * rank            # rank 1 is the slow replica
        worst = replicas.max_over_ranks(local_ms, dist)
        # gather the checksums only to verify (test plumbing; the product path has no such exchange)
        got = [None] * world
        dist.all_gather_object(got, checksum)
        out[rank] = (worst, got, replicas.job_value_ms(worst, 5, world))
    finally:
        dist.destroy_process_group()


def test_two_replicas_gloo():
    world = 2
    port = _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    assert len(out) == world
    for rank in range(world):
        worst, sums, value = out[rank]
        assert worst == 15.0                      # max over ranks, seen by every rank
        assert sums[0] != sums[1]                 # different seeds: different simulations
        assert value == pytest.approx(15.0 / (5 * world))


def test_single_process_is_identity():
    assert replicas.rank_world()[1] >= 1
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.job_value_ms(30.0, 10, 1) == 3.0
