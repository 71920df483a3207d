"""The N > 1 (replica) path on CPU: two gloo ranks agree on max-over-ranks timings and rank 0 aggregates the
whole-job rate; `bench.py --gpus 2` starts its own ranks.  (No GPU: the data path itself has no collective.)"""
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


def test_bench_gpus_2_starts_two_ranks_itself():
    # `python bench.py --gpus 2` without a torchrun environment must start the ranks itself (one process per GPU,
    # rendezvous on 127.0.0.1); exercised on CPU with the reference arm, whose rank 0 prints the line and whose other
    # ranks exit 0 without work
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--impl", "reference", "--steps", "1",
                        "--warmup", "0"], capture_output=True, text=True, timeout=600, env=env, cwd=root)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    out = json.loads(lines[0])
    assert out["impl"] == "reference" and out["n_gpus"] == 2 and out["unit"] == "GB/s"
    assert out["e2e"]["h2d_bytes_per_step"] == 0 and out["cpu_baseline"]["kind"] == "oracle"
