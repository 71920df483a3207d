"""Host logic of the multi-GPU (replica) path.  The hot path shards as independent replicas (DESIGN.md
"Multi-GPU": the paper's rollout workers are data-parallel at TP=1), so there is no
data-path collective: ranks only agree on the timing (max over ranks) and rank 0 reports the whole-job rate."""
from __future__ import annotations

import os


def env_rank_world():
    """(rank, local_rank, world) from the torchrun environment; (0, 0, 1) when launched directly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def max_over_ranks(stats, dist=None, device=None):
    """Element-wise max of a 1-D float64 tensor of durations over all ranks (identity without a process group).
    With NCCL the reduction runs on `device`; with gloo it runs on the CPU tensor itself."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return stats
    t = stats.to(device) if device is not None else stats.clone()
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.cpu()


def whole_job_rate(units_per_rank: float, world: int, ms: float) -> float:
    """Weak scaling over replicas: every rank processed `units_per_rank` in (max over ranks) `ms` milliseconds.
    Returns units per second * 1e-9 when units are bytes (GB/s)."""
    if ms <= 0.0:
        raise ValueError("non-positive duration")
    return units_per_rank * world / ms / 1e6
