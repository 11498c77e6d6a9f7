"""The N>1 path of bench.py on CPU: world_size 2, gloo.  The compress_window path shards by sequence with
no data-path collective, so what is tested is what crosses ranks — per-rank seeds, the
barrier, the max-over-ranks time and the whole-job throughput — plus that two replicas really draw
different batches and that their oracle results are independent of each other."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(world))
    sys.path.insert(0, str(ROOT))
    from paper_2607_01237_b200 import inputs as kin
    from paper_2607_01237_b200 import replicas
    dist.init_process_group("gloo", rank=rank, world_size=world)
    r, lr, w = replicas.rank_env()
    assert (r, lr, w) == (rank, rank, world)
    wl = kin.generate(kin.CFG1, seed=replicas.rank_seed(1, r))
    dist.barrier()
    my_ms = [10.0 + 5.0 * r, 3.0 - r]                 # rank 1 is slower on the first, faster on the second
    mx = replicas.max_over_ranks(my_ms, dist, "cpu")
    dist.barrier()
    value = replicas.job_throughput(w, 8, 4, mx[0])
    # ship this rank's batch fingerprint and results to the parent
    np.save(os.path.join(out_dir, f"q{rank}.npy"), wl.window_q.view(torch.int16).numpy())
    np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array(mx + [value]))
    dist.destroy_process_group()


def test_two_replicas_gloo(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r0, r1 = np.load(tmp_path / "r0.npy"), np.load(tmp_path / "r1.npy")
    np.testing.assert_array_equal(r0, r1)                       # every rank sees the same reduced numbers
    assert r0[0] == 15.0 and r0[1] == 3.0                       # element-wise MAX over ranks
    assert r0[2] == 2 * 8 * 4 / 15e-3                           # whole-job units / slowest rank's time
    q0, q1 = np.load(tmp_path / "q0.npy"), np.load(tmp_path / "q1.npy")
    assert q0.shape == q1.shape and not np.array_equal(q0, q1)  # replicas draw different batches


def test_single_process_is_identity():
    from paper_2607_01237_b200 import replicas
    assert replicas.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert replicas.rank_seed(2, 0) == 2 and replicas.rank_seed(2, 3) == 3002
    assert replicas.job_throughput(1, 40, 10, 2.0) == 40 * 10 / 2e-3


def test_bench_launcher_starts_n_ranks():
    """`bench.py --gpus N` started plainly must start its N ranks itself (replicas.needs_spawn / spawn_ranks): the
    launcher re-executes the script under torch.distributed.run; here with a CPU stand-in for the step (gloo)."""
    import json
    from paper_2607_01237_b200 import replicas
    env_had = os.environ.pop("WORLD_SIZE", None)
    try:
        assert replicas.needs_spawn(2) and not replicas.needs_spawn(1)
        rc, out = replicas.spawn_ranks(2, [str(ROOT / "tests" / "replica_step_cpu.py"), "3"], capture=True)
    finally:
        if env_had is not None:
            os.environ["WORLD_SIZE"] = env_had
    assert rc == 0
    lines = [json.loads(x) for x in out.splitlines() if x.startswith("{")]
    assert len(lines) == 1 and lines[0]["n_gpus"] == 2 and lines[0]["steps"] == 3 and lines[0]["value"] > 0


def test_bench_gpus_n_without_devices_fails_loudly():
    """Fewer CUDA devices than ranks is an error, never a silent N = 1 run."""
    import subprocess
    import pytest
    import torch
    from paper_2607_01237_b200 import replicas
    with pytest.raises(SystemExit):
        replicas.require_devices(2, 1)
    replicas.require_devices(2, 2)
    if torch.cuda.device_count() < 2:
        env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
        r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--gpus", "2", "--steps", "1"], env=env,
                           capture_output=True, text=True)
        assert r.returncode != 0 and "only" in r.stderr and "--gpus 2" in r.stderr
