"""The N > 1 (replica) path on CPU: two gloo ranks agree on max-over-ranks timings and rank 0 aggregates the
whole-job rate; unit sharding is a partition.  (No GPU: the data path itself has no collective.)"""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_18967_b200 import multi


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert multi.env_rank_world() == (rank, rank, world)
        # every rank measured its own durations; the reported ones are the max over ranks
        mine = torch.tensor([1.0 + rank, 5.0 - rank, 2.0], dtype=torch.float64)
        red = multi.max_over_ranks(mine, dist)
        dist.barrier()
        if rank == 0:
            out.put((red.tolist(), multi.whole_job_rate(30.0e6, world, float(red[0]))))
    finally:
        dist.destroy_process_group()


def test_two_ranks_max_timing_and_whole_job_rate():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    red, rate = out.get(timeout=120)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert red == [2.0, 5.0, 2.0]
    assert rate == pytest.approx(30.0e6 * 2 / 2.0 / 1e6)


def test_single_process_is_identity():
    t = torch.tensor([3.0, 1.0], dtype=torch.float64)
    assert torch.equal(multi.max_over_ranks(t, None), t)
    assert multi.whole_job_rate(10.0e6, 1, 2.0) == pytest.approx(5.0)
    with pytest.raises(ValueError):
        multi.whole_job_rate(1.0, 1, 0.0)


@pytest.mark.parametrize("n,world", [(64, 1), (64, 2), (64, 8), (7, 4), (3, 8), (0, 2)])
def test_shard_units_is_a_balanced_partition(n, world):
    ranges = [multi.shard_units(n, r, world) for r in range(world)]
    assert ranges[0][0] == 0 and ranges[-1][1] == n
    assert all(ranges[i][1] == ranges[i + 1][0] for i in range(world - 1))
    sizes = [e - b for b, e in ranges]
    assert max(sizes) - min(sizes) <= 1
