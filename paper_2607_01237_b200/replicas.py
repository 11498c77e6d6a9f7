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


def needs_spawn(n_gpus: int) -> bool:
    """`bench.py --gpus N` started plainly (no torchrun environment) must start its N ranks itself."""
    return n_gpus > 1 and "WORLD_SIZE" not in os.environ


def free_port() -> int:
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def spawn_ranks(n_ranks: int, script_argv, port: int | None = None, capture: bool = False):
    """Re-executes `script_argv` (script path + its arguments) as n_ranks processes of one node through
    torch.distributed.run (one rank per GPU / replica, rendezvous on 127.0.0.1).  Returns its exit code, or
    (exit code, stdout) with capture=True."""
    import subprocess
    import sys
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_ranks}",
           "--master-addr", "127.0.0.1", "--master-port", str(port or free_port()), *script_argv]
    if capture:
        r = subprocess.run(cmd, stdout=subprocess.PIPE, text=True)
        return r.returncode, r.stdout
    return subprocess.call(cmd)


def require_devices(n_ranks: int, available: int) -> None:
    """One replica per GPU: fewer devices than ranks is an error, never a silent N = 1 run."""
    if available < n_ranks:
        raise SystemExit(f"bench.py --gpus {n_ranks}: only {available} CUDA device(s) visible; "
                         "one replica per GPU is required (no oversubscription, no silent fallback to 1)")
