"""CPU stand-in for bench.py's step, started by replicas.spawn_ranks in tests/test_replicas_gloo.py: the same rank
plumbing (rank_env, per-rank seeds, barrier, max-over-ranks time, whole-job throughput, rank 0 prints ONE JSON line)
over gloo, with the CPU generation of a tiny workload as the "step" instead of the CUDA call."""
import json
import sys
import time
from pathlib import Path

import torch.distributed as dist

sys.path.insert(0, str(Path(__file__).resolve().parent.parent))
from paper_2607_01237_b200 import inputs as kin  # noqa: E402
from paper_2607_01237_b200 import replicas  # noqa: E402

rank, local_rank, world = replicas.rank_env()
dist.init_process_group("gloo")
steps = int(sys.argv[1]) if len(sys.argv) > 1 else 2
dist.barrier()
t0 = time.perf_counter()
for i in range(steps):
    wl = kin.generate(kin.CFG1, seed=replicas.rank_seed(1, rank) + i)
ms = (time.perf_counter() - t0) * 1e3
dist.barrier()
(total_ms,) = replicas.max_over_ranks([ms], dist, "cpu")
if rank == 0:
    print(json.dumps({"n_gpus": world, "steps": steps, "value": replicas.job_throughput(world, 1, steps, total_ms),
                      "scaling": "weak"}))
dist.destroy_process_group()
