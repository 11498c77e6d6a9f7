"""Multi-GPU plumbing of bench.py: the path shards with NO exchange — every rank runs an
independent batch (replica) — so all that crosses ranks is the timing: a barrier on both sides of the
timed region and the MAX of the per-rank device times.  Kept here, free of CUDA, so that the world_size-2
gloo tests can run it on CPU."""
from __future__ import annotations

import os


def rank_env():
    """(rank, local_rank, world_size) as torchrun exports them; (0, 0, 1) when launched plainly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def rank_seed(base_seed: int, rank: int) -> int:
    """Each replica gets its own synthetic batch."""
    return base_seed + 1000 * rank


def max_over_ranks(values, dist=None, device="cpu"):
    """Element-wise MAX of a list of floats over all ranks (identity without a process group)."""
    if dist is None:
        return [float(v) for v in values]
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def job_throughput(world: int, units_per_rank_step: float, steps: int, slowest_total_ms: float) -> float:
    """Whole-job units/s: every rank processed units_per_rank_step x steps units in the slowest rank's time."""
    return world * units_per_rank_step * steps / (slowest_total_ms * 1e-3)
