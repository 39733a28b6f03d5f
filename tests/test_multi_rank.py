"""World-size-2 test of the benchmark's multi-rank plumbing on CPU (gloo): the max-over-ranks
timing reduction, the barrier, the view partition and the whole-job aggregate."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2408_12282_b200 import multi


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert multi.env_ranks() == (rank, world, rank)
        multi.barrier()
        local_ms = 10.0 + 5.0 * rank           # rank 1 is the slow one
        worst = multi.max_over_ranks(local_ms)
        views = multi.frames_of_rank(8, rank, world)
        counts = torch.tensor([len(views)], dtype=torch.int64)
        dist.all_reduce(counts)
        multi.barrier()
        q.put((rank, worst, views, int(counts.item())))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [15.0, 15.0]                      # max over ranks on every rank
    assert res[0][2] == [0, 2, 4, 6] and res[1][2] == [1, 3, 5, 7]  # disjoint, complete partition
    assert res[0][3] == 8
    # whole-job aggregate: 2 ranks x 4 steps x 3 frames x 1e6 px in 15 ms
    assert multi.whole_job_mpix_per_s(2, 4, 3, 1_000_000, 15.0) == pytest.approx(2 * 4 * 3 * 1e6 / 15e-3 / 1e6)


def test_single_rank_is_passthrough():
    assert multi.max_over_ranks(3.5) == 3.5
    assert multi.frames_of_rank(5, 0, 1) == [0, 1, 2, 3, 4]
    multi.barrier()
