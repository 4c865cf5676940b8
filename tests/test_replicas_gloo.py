"""N > 1 path of bench.py on CPU: two `gloo` ranks, replicas only (no data-path collective).
Checks the max-over-ranks timing, the whole-job value and that replica seeds never collide."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_19729_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert replicas.env_rank_world() == (rank, rank, world)
    my_ms = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
    worst = replicas.max_over_ranks(my_ms, dist)
    value = replicas.whole_job_value(1000.0, world, worst)
    dist.barrier()
    q.put((rank, worst, value))
    dist.destroy_process_group()


def test_two_replicas_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, worst, value in res:
        assert worst == 15.0                       # the maximum, on every rank
        assert value == pytest.approx(2 * 1000.0 / 15e-3)


def test_single_process_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.whole_job_value(10.0, 1, 2.0) == pytest.approx(5000.0)
    assert replicas.env_rank_world()[2] >= 1


def test_replica_seeds_distinct():
    seen = set()
    for rank in range(8):
        for step in range(50):
            for call in (0, 1):
                seen.add(replicas.replica_seed(20260619, rank, step, call))
    assert len(seen) == 8 * 50 * 2
    assert replicas.replica_seed(20260619, 0, 3, 1) == 20260619 + 7
