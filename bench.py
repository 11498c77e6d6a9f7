#!/usr/bin/env python
"""bench.py — Kara compress_window step on B200: window-compressions/s, KV GB/s, % of roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload cfg2|cfg3|cfg4|cfg5|cfg1]

A "step" is ONE pass of the whole hot path (a1 score, a2 top-k, a3 Token2Chunk, a4 compaction,
a5 metadata) over one batch of synthetic input: one kara_compress_window call over all resident
layers with KARA_COMMIT.  Default workload = BASELINE.json configs[1] (single sequence,
Qwen3-14B-like 40 layers x 40/8 heads x 128, h=4096, W=512, U=32, r=20 %, alpha=32, gamma=8).
The call is destructive, so between steps the pools / tables / free list are restored from a
pristine copy and L2 is flushed (both untimed); every step is timed on its own with CUDA events
on the launching stream, and the K step times are summed (max over ranks for N>1).

Prints ONE JSON line (see DESIGN.md §Measurement for every key).  `--impl reference` times the
CPU oracle, as it stands, on a bounded sample of the same workload (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "window-compressions/sec"
UNIT = "window-compressions/s"


def _shape(name):
    from paper_2607_01237_b200 import inputs as kin
    table = {"cfg1": kin.CFG1, "cfg2": kin.CFG2, "cfg3": kin.CFG3, "cfg4": kin.CFG4, "cfg5": kin.CFG5}
    return table[name]


def _resident_layers(name, shape, requested):
    if requested:
        return requested
    # SURVEY §8(d) footprint: cfg 3 fits with all layers only barely, cfg 4/5 do not fit at all
    return {"cfg3": 8, "cfg4": 2, "cfg5": 8}.get(name, shape.n_layers)


def _config(name, shape, L, extra=None):
    cfg = {"workload": f"BASELINE.json configs[{int(name[-1]) - 1}] ({shape.name})",
           "n_seqs": shape.n_seqs, "n_layers": L, "n_layers_model": shape.n_layers,
           "n_q_heads": shape.n_q_heads, "n_kv_heads": shape.n_kv_heads, "head_dim": shape.head_dim,
           "block_size": shape.block_size, "W": shape.W, "U": shape.U, "retention": shape.ratio,
           "alpha": shape.alpha, "gamma": shape.gamma, "history": [shape.hist_lo, shape.hist_hi],
           "query_mean_shift_c": shape.q_shift, "key_dist": shape.k_dist,
           "l2": "flushed between steps (256 MiB write); per-step inputs (Q + window KV) exceed L2 at cfg2+",
           "timing": "per-step CUDA events on the launching stream; state restore + L2 flush between steps untimed",
           "parallelism": "replicas (one independent batch per GPU, no collective)"}
    cfg.update(extra or {})
    return cfg


def algorithmic(shape, L):
    """Algorithmic FLOPs and bytes of one step."""
    import math
    n = shape.n
    keep = int(math.ceil(shape.ratio * n - 1e-9))
    units = shape.n_seqs * L * shape.n_kv_heads
    flops_unit = 2.0 * shape.W * shape.G * n * shape.head_dim
    q_bytes = shape.W * shape.G * shape.head_dim * 2
    k_bytes = n * shape.head_dim * 2
    comp_bytes = 2 * 2 * (keep + shape.U) * shape.head_dim * 2     # K and V, read + write
    return dict(units=units, keep=keep, flops_unit=flops_unit, bytes_unit=q_bytes + k_bytes + comp_bytes,
                flops=flops_unit * units, bytes=(q_bytes + k_bytes + comp_bytes) * units,
                kv_in_bytes=shape.n_seqs * L * shape.W * shape.n_kv_heads * shape.head_dim * 2 * 2)


# dram__bytes_read.sum + dram__bytes_write.sum of ONE score-kernel launch from the committed `ncu --set full`
# capture (profiles/r1_final_ncu_cfg2.md), keyed by (workload, resident layers); None where no capture exists.
NCU_SCORE_TRAFFIC_BYTES = {("cfg2", 40): 257.7e6 + 6.7e6}


def _peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        j = json.loads(p.read_text())
        return dict(hbm_gbs=j["hbm_gbs"], bf16_tflops=j["bf16_tflops"],
                    bf16_tflops_sustained=j.get("bf16_tflops_sustained"), source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0,
                source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """Samples SM clock and throttle reasons DURING the timed region (pynvml, else nvidia-smi)."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown"}

    def __init__(self, index):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._ready = threading.Event()
        self._t = None

    def _loop(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = int(vis.split(",")[self.index]) if vis and vis.split(",")[self.index].isdigit() else self.index
            h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
            while not self._stop.is_set():
                self.samples.append(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                r = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, nm in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(nm)
                self._ready.set()
                time.sleep(0.005)
        except Exception as e:  # noqa: BLE001
            self.reasons.add(f"sampler_error:{type(e).__name__}")
            self._ready.set()

    def __enter__(self):
        self._t = threading.Thread(target=self._loop, daemon=True)
        self._t.start()
        self._ready.wait(timeout=10)      # NVML is initialised and sampling before the timed region starts
        self.samples.clear()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=2)

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


# -------------------------------------------------------------------------------------------------
def oracle_prepare(shape, L_sample, seed):
    """Host image of `L_sample` layers of the workload's first sequence for the oracle legs."""
    from oracle import check
    from paper_2607_01237_b200 import inputs as kin
    small = kin.scaled(shape, n_seqs=1, n_layers=L_sample, hist_lo=min(shape.hist_lo, 4096),
                       hist_hi=min(shape.hist_lo, 4096))
    wl = kin.generate(small, seed=seed)
    desc = (f"{L_sample} layer(s) x 1 sequence x {small.n_kv_heads} KV heads = {L_sample * small.n_kv_heads} units of "
            f"{shape.name} (whole path O1-O11, fp64, 1 thread); history capped at 4096 tokens (never read)")
    return small, check.host_image(wl), desc


def oracle_leg(small, H, L_sample):
    """One timed pass of the CPU oracle, as it stands (1 thread), over the prepared sample."""
    from oracle import check
    Hc = {k: v.copy() for k, v in H.items()}
    t0 = time.perf_counter()
    check.run_oracle(Hc, small.n_q_heads, small.W, small.U, small.ratio, small.alpha, small.gamma, 0, L_sample)
    return time.perf_counter() - t0


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    shape = _shape(args.workload)
    L_sample = 1     # one layer of one sequence per step (cfg 2: 8 units, about 1.2 s)
    small, H, desc = oracle_prepare(shape, L_sample, seed=2)
    for _ in range(args.warmup):
        oracle_leg(small, H, L_sample)
    times = [oracle_leg(small, H, L_sample) for _ in range(args.steps)]
    total = sum(times)
    value = L_sample * args.steps / total
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": _config(args.workload, shape, L_sample, {"sample": desc}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# -------------------------------------------------------------------------------------------------
def run_gpu(args):
    import torch
    from paper_2607_01237_b200 import inputs as kin
    from paper_2607_01237_b200 import kara
    from paper_2607_01237_b200 import replicas

    rank, local_rank, world = replicas.rank_env()
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    torch.cuda.set_device(local_rank)
    dev = torch.device(f"cuda:{local_rank}")
    kara.lib()

    shape = _shape(args.workload)
    L = _resident_layers(args.workload, shape, args.layers)
    seed = replicas.rank_seed({"cfg1": 1, "cfg2": 2, "cfg3": 3, "cfg4": 4, "cfg5": 5}[args.workload], rank)
    fill = "randn" if args.workload in ("cfg1", "cfg2") else "pattern"
    wl = kin.generate(shape, seed=seed, device=dev, n_layers_resident=L, history_fill=fill)
    alg = algorithmic(shape, L)
    peaks = _peaks()

    cache = kara.KaraCache(shape.block_size, L, shape.n_kv_heads, shape.head_dim)
    cache.attach_pool(wl.k_pool, wl.v_pool, wl.free_list, wl.free_count)
    cache.enable_score_timing(not args.no_score_timing)
    flags = kara.KARA_COMMIT | (kara.KARA_SCORE_SIMT if args.simt else 0)
    ws = torch.empty(cache.workspace_bytes(L, shape.n_seqs, shape.n_q_heads, shape.W, shape.U, shape.ratio,
                                           shape.alpha), dtype=torch.uint8, device=dev)
    # pristine copies: only the window blocks change, but a full copy is simple and untimed
    if wl.k_pool.numel() * 2 <= 8 << 30:
        k0, v0 = wl.k_pool.clone(), wl.v_pool.clone()
        win_blocks = None
    else:   # large pools: save / restore just the blocks the windows touch
        bs = shape.block_size
        ids = []
        for s in range(shape.n_seqs):
            h, ln = int(wl.win_start[s]), int(wl.seq_lens[s])
            ids.append(wl.block_table[s, h // bs:(ln + bs - 1) // bs])
        win_blocks = torch.cat(ids).long()
        k0, v0 = wl.k_pool[:, win_blocks].clone(), wl.v_pool[:, win_blocks].clone()
    bt0, sl0, fl0, fc0 = wl.block_table.clone(), wl.seq_lens.clone(), wl.free_list.clone(), wl.free_count.clone()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def restore():
        if win_blocks is None:
            wl.k_pool.copy_(k0); wl.v_pool.copy_(v0)
        else:
            wl.k_pool[:, win_blocks] = k0; wl.v_pool[:, win_blocks] = v0
        wl.block_table.copy_(bt0); wl.seq_lens.copy_(sl0); wl.free_list.copy_(fl0); wl.free_count.copy_(fc0)
        flush.zero_()
        torch.cuda.synchronize()

    def step():
        cache.compress_window(0, L, wl.block_table, wl.seq_lens, wl.win_start, wl.window_q, shape.W, shape.U,
                              shape.ratio, shape.alpha, shape.gamma, flags, workspace=ws)

    stream = torch.cuda.current_stream(dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(args.warmup):
        restore(); step(); torch.cuda.synchronize()
    assert cache.status() == 0, "device status word set during warm-up"
    freed = int(wl.free_count[0]) - int(fc0[0])

    step_ms, score_ms = [], []
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    with ClockSampler(local_rank) as clk:
        for _ in range(args.steps):
            restore()
            ev0.record(stream); step(); ev1.record(stream)
            torch.cuda.synchronize()
            step_ms.append(ev0.elapsed_time(ev1))
            score_ms.append(cache.score_kernel_ms())
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    launches = cache.last_launch_count() * args.steps
    score_path = cache.last_score_path()
    total_ms = sum(step_ms)

    # ---- e2e: same step through the host-buffer entry point (pinned host inputs) -------------
    hq = wl.window_q.cpu().pin_memory()
    hbt, hsl, hws = bt0.cpu().pin_memory(), sl0.cpu().pin_memory(), wl.win_start.cpu().pin_memory()
    h2d = hq.numel() * 2 + hbt.numel() * 4 + hsl.numel() * 4 + hws.numel() * 4
    d2h = hbt.numel() * 4 + hsl.numel() * 4 + 4
    e2e_s = []
    n_e2e = max(3, min(args.steps, 10))
    for it in range(2 + n_e2e):
        restore()
        hbt.copy_(bt0.cpu()); hsl.copy_(sl0.cpu())
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        cache.compress_window_host(0, L, hbt, hsl, hws, hq, shape.W, shape.U, shape.ratio, shape.alpha, shape.gamma,
                                   flags)
        dt = time.perf_counter() - t0
        if it >= 2:
            e2e_s.append(dt)
    e2e_total = sum(e2e_s)

    total_ms, e2e_mean = replicas.max_over_ranks([total_ms, e2e_total / len(e2e_s)], dist, dev)

    wc_step = shape.n_seqs * L                      # window-compressions per step per GPU
    value = replicas.job_throughput(world, wc_step, args.steps, total_ms)
    ms_per_step = total_ms / args.steps
    sc_ms = sum(score_ms) / len(score_ms)
    t_tensor_ms = alg["flops"] / (peaks["bf16_tflops"] * 1e12) * 1e3
    t_hbm_ms = alg["bytes"] / (peaks["hbm_gbs"] * 1e9) * 1e3
    achieved_tflops = alg["flops"] / (sc_ms * 1e-3) / 1e12

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": _config(args.workload, shape, L, {"score_kernel": {1: "simt", 2: "tcgen05+tma"}.get(score_path),
                                                     "freed_blocks_per_step": freed}),
        "kv_gbs": world * alg["kv_in_bytes"] / (ms_per_step * 1e-3) / 1e9,
        "algorithmic_gbs": world * alg["bytes"] / (ms_per_step * 1e-3) / 1e9,
        "step_tflops": world * alg["flops"] / (ms_per_step * 1e-3) / 1e12,
        "clocks": clk.summary(),
        "e2e": {"value": world * wc_step / e2e_mean, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": e2e_mean * 1e3,
                "api": "kara_compress_window_host (pinned host window_q/tables in, tables + free count out)"},
        "gpu_launches": launches,
        "roofline": {"kernel": "score (a1)", "bound": "tensor", "achieved": achieved_tflops,
                     "peak": peaks["bf16_tflops"], "unit": "TFLOP/s", "frac": achieved_tflops / peaks["bf16_tflops"],
                     "traffic": NCU_SCORE_TRAFFIC_BYTES.get((args.workload, L)),
                     "traffic_source": "profiles/r1_final_ncu_cfg2.md (ncu --set full, dram rd+wr of one launch)",
                     "peak_source": peaks["source"] + ", burst bf16", "kernel_ms": sc_ms,
                     "flops_per_launch": alg["flops"], "share_of_step": sc_ms / ms_per_step},
        "step_roofline": {"t_tensor_ms": t_tensor_ms, "t_hbm_ms": t_hbm_ms,
                          "frac": max(t_tensor_ms, t_hbm_ms) / ms_per_step,
                          "def": "slower of (algorithmic bytes / measured HBM GB/s) and (score FLOPs / measured bf16 TFLOP/s) over ms_per_step"},
    }
    if rank == 0:
        if not args.no_cpu_baseline and world == 1:
            Ls = {"cfg1": 1, "cfg2": 24, "cfg3": 24, "cfg4": 6, "cfg5": 2}[args.workload]   # ~10-30 s of CPU work
            small, H, desc = oracle_prepare(shape, Ls, seed=2)
            secs = oracle_leg(small, H, Ls)
            import multiprocessing
            line["cpu_baseline"] = {"value": Ls / secs, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc,
                                    "seconds": secs, "host_cores_available": multiprocessing.cpu_count()}
        print(json.dumps(line))
    if dist:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--layers", type=int, default=0, help="resident layers (default: all that fit)")
    ap.add_argument("--simt", action="store_true", help="force the CUDA-core score kernel")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-score-timing", action="store_true",
                    help="no CUDA events inside the library around the score launch (roofline.kernel_ms = 0)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
