"""world_size-2 gloo test (CPU) of the N>1 bookkeeping bench.py uses: replicas only, no data-path collective."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1803_01190_b200 import replicas, workloads


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert replicas.env_rank() == (rank, rank, world)
        seed = replicas.replica_seed(2, rank)
        pos, _, _ = workloads.make("disk", 64, seed)
        replicas.barrier()
        ms_local = 100.0 + 50.0 * rank                  # rank 1 is the slow one
        ms = replicas.max_over_ranks(ms_local)
        out[rank] = (seed, float(pos[0, 0]), ms, replicas.job_value(64 * 63, 5, ms, world))
    finally:
        dist.destroy_process_group()


def test_two_replicas_distinct_inputs_and_max_time():
    world = 2
    mgr = mp.get_context("spawn").Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    (s0, x0, ms0, v0), (s1, x1, ms1, v1) = out[0], out[1]
    assert s0 == 2 and s1 == 1002 and x0 != x1          # independent systems
    assert ms0 == ms1 == 150.0                          # max over ranks, seen by every rank
    assert v0 == v1 == pytest.approx(2 * 64 * 63 * 5 / 0.150)


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.job_value(10, 2, 1000.0, 1) == 20.0
    replicas.barrier()
