#!/usr/bin/env python
"""bench.py — Kara compress_window step on B200: window-compressions/s, KV GB/s, % of roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
                    [--workload cfg4|cfg2|cfg3|cfg5|cfg1|prefill] [--qbuf-only] [--alpha0] [--no-per-config]

A "step" is ONE pass of the whole hot path (a1 score, a2 top-k, a3 Token2Chunk, a4 compaction,
a5 metadata) over one batch of synthetic input: one kara_compress_window call over all resident
layers with KARA_COMMIT.  Default workload = BASELINE.json configs[3] (cfg4: 256 concurrent
sequences, Qwen3-14B-like 40/8 heads x 128, W=1024, U=32, r=20 %, alpha=32, gamma=8, histories in
[8K, 32K], pool 95 % full; 2 of 40 layers resident — 40 layers do not fit 180 GB), the
largest single-GPU configuration of the metric.  The same JSON line carries `per_config`: cfg2, cfg3,
cfg5 and the prefill workload, a few steps each.
The call is destructive, so between steps the pools / tables / free list are restored from a
pristine copy and L2 is flushed (both untimed); every step is timed on its own with CUDA events
on the launching stream, and the K step times are summed (max over ranks for N>1).

`--gpus N` without a torchrun environment starts its N ranks itself (one replica per GPU, no
data-path collective: DESIGN.md §8) and fails loudly if fewer than N devices are visible.
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
WORKLOADS = ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "prefill")
SEEDS = {"cfg1": 1, "cfg2": 2, "cfg3": 3, "cfg4": 4, "cfg5": 5, "prefill": 6}


def _shape(name):
    from paper_2607_01237_b200 import inputs as kin
    table = {"cfg1": kin.CFG1, "cfg2": kin.CFG2, "cfg3": kin.CFG3, "cfg4": kin.CFG4, "cfg5": kin.CFG5,
             "prefill": kin.PREFILL}
    return table[name]


def _resident_layers(name, shape, requested):
    if requested:
        return requested
    # SURVEY §8(d) footprint: cfg 3 fits with all layers only barely, cfg 4/5 do not fit at all
    return {"cfg3": 8, "cfg4": 2, "cfg5": 8, "prefill": 8}.get(name, shape.n_layers)


def _workload_label(name, shape):
    if name == "prefill":
        return f"SURVEY 8(f)-1 prefill ({shape.name}: {shape.n_seqs} prompts x {shape.n_windows} windows of {shape.W})"
    return f"BASELINE.json configs[{int(name[-1]) - 1}] ({shape.name})"


def _config(name, shape, L, extra=None):
    cfg = {"workload": _workload_label(name, shape),
           "n_seqs": shape.n_seqs, "n_windows": shape.n_windows, "n_layers": L, "n_layers_model": shape.n_layers,
           "n_q_heads": shape.n_q_heads, "n_kv_heads": shape.n_kv_heads, "head_dim": shape.head_dim,
           "block_size": shape.block_size, "W": shape.W, "U": shape.U, "retention": shape.ratio,
           "alpha": shape.alpha, "gamma": shape.gamma, "history": [shape.hist_lo, shape.hist_hi],
           "query_mean_shift_c": shape.q_shift, "key_dist": shape.k_dist,
           "l2": "flushed between steps (256 MiB write); per-step inputs (Q + window KV) exceed L2 at cfg2+",
           "timing": "per-step CUDA events on the launching stream; state restore + L2 flush between steps untimed",
           "parallelism": "replicas (one independent batch per GPU, no collective)"}
    cfg.update(extra or {})
    return cfg


def algorithmic(shape, L, qbuf_only=False):
    """Algorithmic FLOPs and bytes of one step.  A window-compression is
    one (sequence, layer, window) over all KV heads; with --qbuf-only the queries are the U buffer rows."""
    import math
    n = shape.n
    keep = int(math.ceil(shape.ratio * n - 1e-9))
    units = shape.n_seqs * shape.n_windows * L * shape.n_kv_heads
    q_rows = shape.U if qbuf_only else shape.W
    flops_unit = 2.0 * q_rows * shape.G * n * shape.head_dim
    q_bytes = q_rows * shape.G * shape.head_dim * 2
    k_bytes = n * shape.head_dim * 2
    comp_bytes = 2 * 2 * (keep + shape.U) * shape.head_dim * 2     # K and V, read + write
    return dict(units=units, keep=keep, flops_unit=flops_unit, bytes_unit=q_bytes + k_bytes + comp_bytes,
                flops=flops_unit * units, bytes=(q_bytes + k_bytes + comp_bytes) * units,
                score_bytes=(q_bytes + k_bytes) * units,
                kv_in_bytes=shape.n_seqs * shape.n_windows * L * shape.W * shape.n_kv_heads * shape.head_dim * 2 * 2)


# dram__bytes_read.sum + dram__bytes_write.sum of ONE score-kernel launch, from the committed `ncu --set full`
# captures of exactly these commands, keyed by (workload, resident layers, variant): cfg4 from the round-3 capture
# (profiles/r3_ncu.md, commit 0e978c3), the others from round 2's (profiles/r2_ncu_score.md, commit 26d0175 — the score
# kernel's SASS has not changed since).
NCU_SCORE_TRAFFIC_BYTES = {("cfg2", 40, "full"): 257.957e6 + 4.504e6, ("cfg3", 8, "full"): 3212.377e6 + 20.670e6,
                           ("cfg4", 2, "full"): 6434.983e6 + 30.275e6, ("cfg5", 8, "full"): 4827.730e6 + 32.882e6,
                           ("cfg4", 2, "qbuf_only"): 1229.311e6 + 19.162e6}
NCU_TRAFFIC_SOURCE = ("profiles/r3_ncu.md for cfg4, profiles/r2_ncu_score.md for the other workloads "
                      "(ncu --set full, dram rd+wr of one score-kernel launch of this workload)")
# The number is only reported while the score kernel's sources are still the ones the captures describe (sha256 over the
# files below, in this order) — otherwise `traffic` is null and `traffic_stale` true.
NCU_TRAFFIC_COMMIT = "0e978c3 (cfg4) / 26d0175 (others)"
SCORE_KERNEL_SOURCES = ("score_tc.cu", "score_tc_ptx.cuh", "score_tc.h")
# (the sources of commit 0e978c3, the round-3 capture's; the round-2 captures predate the removal of the trace / diagnostic
# switches and of unused PTX helpers, which left `cuobjdump -sass` of score_tc.o identical instruction for instruction)
SCORE_KERNEL_SHA256_AT_CAPTURE = "766c3e9f98689d782663db473fe64f64d42b572f55dc1a68844662c106551abe"


def score_kernel_sha256():
    import hashlib
    h = hashlib.sha256()
    for f in SCORE_KERNEL_SOURCES:
        h.update((ROOT / "paper_2607_01237_b200" / "csrc" / f).read_bytes())
    return h.hexdigest()


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
# CPU oracle legs (cpu_baseline, --impl reference): the oracle as it stands, never tuned for this
def oracle_prepare(shape, L_sample, seed):
    """Host image of `L_sample` layers of the workload's first sequence for the oracle legs."""
    from oracle import check
    from paper_2607_01237_b200 import inputs as kin
    small = kin.scaled(shape, n_seqs=1, n_layers=L_sample, hist_lo=min(shape.hist_lo, 4096),
                       hist_hi=min(shape.hist_lo, 4096))
    wl = kin.generate(small, seed=seed)
    units = L_sample * small.n_windows * small.n_kv_heads
    desc = (f"{L_sample} layer(s) x 1 sequence x {small.n_windows} window(s) x {small.n_kv_heads} KV heads = {units} "
            f"units of {shape.name} (whole path O1-O11, fp64, 1 thread per process); history capped at 4096 tokens "
            f"(never read)")
    return small, check.host_image(wl), desc


def oracle_leg(small, H, L_sample):
    """One timed pass of the CPU oracle, as it stands (1 thread), over the prepared sample."""
    from oracle import check
    Hc = {k: v.copy() for k, v in H.items()}
    t0 = time.perf_counter()
    check.run_oracle(Hc, small.n_q_heads, small.W, small.U, small.ratio, small.alpha, small.gamma, 0, L_sample,
                     n_windows=small.n_windows)
    return time.perf_counter() - t0


def _oracle_worker(args):
    """One process of the all-cores leg: its own sample (a different seed per process), a barrier so that all
    processes run the oracle at the same time, then one timed pass.  Returns (start, end) wall-clock stamps."""
    workload, L_sample, seed, barrier = args
    sys.path.insert(0, str(ROOT))
    small, H, _ = oracle_prepare(_shape(workload), L_sample, seed)
    from oracle import check
    barrier.wait()
    t0 = time.time()
    check.run_oracle(H, small.n_q_heads, small.W, small.U, small.ratio, small.alpha, small.gamma, 0, L_sample,
                     n_windows=small.n_windows)
    return t0, time.time()


def oracle_all_cores(workload, L_per_proc):
    """Independent units in one worker process per core of sched_getaffinity (process-level parallelism, no shared
    code with the GPU path): window-compressions of all processes / (last end - first start)."""
    import multiprocessing as mp
    cores = len(os.sched_getaffinity(0))
    ctx = mp.get_context("spawn")
    with ctx.Manager() as mgr:
        barrier = mgr.Barrier(cores)
        with ctx.Pool(cores) as pool:
            stamps = pool.map(_oracle_worker, [(workload, L_per_proc, 100 + i, barrier) for i in range(cores)])
    wall = max(e for _, e in stamps) - min(s for s, _ in stamps)
    shape = _shape(workload)
    return cores, cores * L_per_proc * shape.n_windows / wall, wall


# layers of one sequence per oracle pass: about 10-30 s of CPU work on one core
ORACLE_LAYERS = {"cfg1": 1, "cfg2": 24, "cfg3": 24, "cfg4": 8, "cfg5": 2, "prefill": 2}   # cfg4: 8 layers x 8 heads = 64 units
ORACLE_LAYERS_PER_PROC = {"cfg1": 1, "cfg2": 8, "cfg3": 8, "cfg4": 2, "cfg5": 1, "prefill": 1}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    shape = _shape(args.workload)
    L_sample = 1     # one layer of one sequence per step (cfg 4: 8 units, about 2 s)
    small, H, desc = oracle_prepare(shape, L_sample, seed=2)
    for _ in range(args.warmup):
        oracle_leg(small, H, L_sample)
    times = [oracle_leg(small, H, L_sample) for _ in range(args.steps)]
    total = sum(times)
    value = L_sample * small.n_windows * args.steps / total
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": _config(args.workload, shape, L_sample, {"sample": desc}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# -------------------------------------------------------------------------------------------------
def measure(name, L_req, steps, warmup, dev, rank, dist, local_rank, simt=False, qbuf_only=False, alpha0=False,
            score_timing=True, want_e2e=False, ratio=None, per_layer_calls=False, also_without_events=False,
            want_chain=False):
    """Generates workload `name` on `dev`, times `steps` steps (after `warmup`) and returns the raw numbers.
    ratio: retention override (BASELINE.json configs[3] sweeps 10 / 20 / 30 %).  per_layer_calls: the step is one
    kara_compress_window call PER LAYER (KARA_COMMIT on the last), the way Alg. 1 l.6-12 interleaves with the model's
    layers, instead of one call over all resident layers.  also_without_events: `steps` more steps with the library's
    event pair around the score launch switched off (the select kernel is launched programmatically behind the score
    kernel; an event record between the two sits where that overlap happens)."""
    import torch
    from paper_2607_01237_b200 import inputs as kin
    from paper_2607_01237_b200 import kara
    from paper_2607_01237_b200 import replicas

    shape = _shape(name)
    if alpha0:
        shape = kin.scaled(shape, alpha=0)                   # "w/o Token2Chunk"
    if ratio is not None:
        shape = kin.scaled(shape, ratio=ratio)
    L = _resident_layers(name, shape, L_req)
    NW = shape.n_windows
    seed = replicas.rank_seed(SEEDS[name], rank)
    fill = "randn" if name in ("cfg1", "cfg2") else "pattern"
    wl = kin.generate(shape, seed=seed, device=dev, n_layers_resident=L, history_fill=fill)

    cache = kara.KaraCache(shape.block_size, L, shape.n_kv_heads, shape.head_dim)
    cache.attach_pool(wl.k_pool, wl.v_pool, wl.free_list, wl.free_count)
    cache.enable_score_timing(score_timing)
    flags = kara.KARA_COMMIT | (kara.KARA_SCORE_SIMT if simt else 0) | (kara.KARA_SCORE_QBUF_ONLY if qbuf_only else 0)
    ws = torch.empty(cache.workspace_bytes(L, shape.n_seqs * NW, shape.n_q_heads, shape.W, shape.U, shape.ratio,
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
        if per_layer_calls:
            for l in range(L):
                cache.compress_window(l, l + 1, wl.block_table, wl.seq_lens, wl.win_start, wl.window_q[l:l + 1], shape.W,
                                      shape.U, shape.ratio, shape.alpha, shape.gamma,
                                      flags if l == L - 1 else flags & ~kara.KARA_COMMIT, workspace=ws)
        elif NW > 1:
            cache.compress_windows(0, L, wl.block_table, wl.seq_lens, wl.win_start, NW, wl.window_q, shape.W, shape.U,
                                   shape.ratio, shape.alpha, shape.gamma, flags, workspace=ws)
        else:
            cache.compress_window(0, L, wl.block_table, wl.seq_lens, wl.win_start, wl.window_q, shape.W, shape.U,
                                  shape.ratio, shape.alpha, shape.gamma, flags, workspace=ws)

    stream = torch.cuda.current_stream(dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(warmup):
        restore(); step(); torch.cuda.synchronize()
    assert cache.status() == 0, "device status word set during warm-up"
    freed = int(wl.free_count[0]) - int(fc0[0])
    score_path = cache.last_score_path()
    if score_path != 2 and not simt:
        # north_star: no multi-backend dispatch — a bench number from the CUDA-core kernel is not a bench number
        raise SystemExit(f"bench.py: workload {name} did not run on the tcgen05/TMA score kernel "
                         f"(kara_last_score_path = {score_path}: {cache.last_score_path_reason()}); pass --simt to time the "
                         "CUDA-core kernel on purpose")

    step_ms, score_ms = [], []
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    with ClockSampler(local_rank) as clk:
        for _ in range(steps):
            restore()
            ev0.record(stream); step(); ev1.record(stream)
            torch.cuda.synchronize()
            step_ms.append(ev0.elapsed_time(ev1))
            score_ms.append(cache.score_kernel_ms())
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    launches_step = cache.last_launch_count() if not per_layer_calls else 2 * L + 1   # (score + select) per layer + a5
    res = dict(shape=shape, L=L, total_ms=sum(step_ms), score_ms=sum(score_ms) / len(score_ms), freed=freed,
               launches=launches_step * steps, score_path=score_path, clocks=clk.summary(),
               alg=algorithmic(shape, L, qbuf_only), wc_step=shape.n_seqs * NW * L, e2e=None, ms_no_events=None)
    if also_without_events:
        cache.enable_score_timing(False)
        ms = []
        for it in range(2 + steps):
            restore()
            ev0.record(stream); step(); ev1.record(stream)
            torch.cuda.synchronize()
            if it >= 2:
                ms.append(ev0.elapsed_time(ev1))
        res["ms_no_events"] = sum(ms) / len(ms)
        cache.enable_score_timing(score_timing)

    # ---- e2e: same step through the host-buffer entry point (pinned host inputs) -------------
    if want_e2e and NW == 1:
        hq = wl.window_q.cpu().pin_memory()
        hbt, hsl, hws = bt0.cpu().pin_memory(), sl0.cpu().pin_memory(), wl.win_start.cpu().pin_memory()
        h2d = hq.numel() * 2 + hbt.numel() * 4 + hsl.numel() * 4 + hws.numel() * 4
        d2h = hbt.numel() * 4 + hsl.numel() * 4 + 4
        e2e_s = []
        n_e2e = max(3, min(steps, 10))
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
        res["e2e"] = dict(mean_s=sum(e2e_s) / len(e2e_s), h2d=h2d, d2h=d2h)
        del hq
    # ---- device-resident chain: hidden states -> kara_window_queries -> kara_compress_window, layer by layer -------
    # What a serving engine runs at a compression event (App. C.2: the window's query states are
    # recomputed on the device; they never cross PCIe): per resident layer the window-query producer writes window_q[l]
    # from the layer's hidden states, then that layer is compressed (KARA_COMMIT on the last).  Synthetic hidden states
    # (one [n_seqs*W, d_model] bf16 buffer shared by the layers) and per-layer random W_q at the model's d_model =
    # n_q_heads * head_dim; positions = the window tokens' own.  The producer goes through the no-allocation entry point.
    res["chain"] = None
    if want_chain and NW == 1:
        Hq, d = shape.n_q_heads, shape.head_dim
        Dm, T = Hq * d, shape.n_seqs * shape.W
        hid = torch.randn(T, Dm, device=dev, dtype=torch.bfloat16)
        wqs = [(torch.randn(Hq * d, Dm, device=dev, dtype=torch.bfloat16) / Dm ** 0.5) for _ in range(L)]
        pos = (wl.win_start.view(-1, 1) + torch.arange(shape.W, device=dev, dtype=torch.int32).view(1, -1)).reshape(-1)
        pos = pos.to(torch.int32).contiguous()
        max_pos = int(pos.max())
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(L)]
        cache.enable_score_timing(False)
        chain_ms, prod_ms = [], []
        n_chain = max(3, min(steps, 10))
        for it in range(2 + n_chain):
            restore()
            ev0.record(stream)
            for l in range(L):
                evs[l][0].record(stream)
                kara.kara_window_queries_static(hid, wqs[l], pos, 1e6, Hq, d, wl.window_q[l].view(T, Hq, d), max_pos)
                evs[l][1].record(stream)
                cache.compress_window(l, l + 1, wl.block_table, wl.seq_lens, wl.win_start, wl.window_q[l:l + 1], shape.W,
                                      shape.U, shape.ratio, shape.alpha, shape.gamma,
                                      flags if l == L - 1 else flags & ~kara.KARA_COMMIT, workspace=ws)
            ev1.record(stream)
            torch.cuda.synchronize()
            if it >= 2:
                chain_ms.append(ev0.elapsed_time(ev1))
                prod_ms.append(sum(evs[l][0].elapsed_time(evs[l][1]) for l in range(L)))
        assert cache.status() == 0, "device status word set in the chain leg"
        res["chain"] = dict(ms=sum(chain_ms) / len(chain_ms), producer_ms=sum(prod_ms) / len(prod_ms), steps=n_chain,
                            hidden_bytes=hid.numel() * 2, d_model=Dm, tokens=T,
                            producer_flops=2.0 * T * Dm * Hq * d * L, launches=(2 + 2) * L + 1)
        del hid, wqs, pos
    cache.close()
    del wl, k0, v0, ws, flush, cache
    torch.cuda.empty_cache()
    return res


def derived(res, peaks, world=1, total_ms=None, steps=1):
    """Throughput and roofline figures of one measure() result (total_ms: max over ranks if given)."""
    alg = res["alg"]
    ms_per_step = (total_ms if total_ms is not None else res["total_ms"]) / steps
    sc_ms = res["score_ms"]
    t_tensor_ms = alg["flops"] / (peaks["bf16_tflops"] * 1e12) * 1e3
    t_hbm_ms = alg["bytes"] / (peaks["hbm_gbs"] * 1e9) * 1e3
    return dict(ms_per_step=ms_per_step, value=world * res["wc_step"] / (ms_per_step * 1e-3),
                kv_gbs=world * alg["kv_in_bytes"] / (ms_per_step * 1e-3) / 1e9,
                algorithmic_gbs=world * alg["bytes"] / (ms_per_step * 1e-3) / 1e9,
                step_tflops=world * alg["flops"] / (ms_per_step * 1e-3) / 1e12,
                score_ms=sc_ms, score_tflops=alg["flops"] / (sc_ms * 1e-3) / 1e12 if sc_ms > 0 else None,
                score_gbs=alg["score_bytes"] / (sc_ms * 1e-3) / 1e9 if sc_ms > 0 else None,
                t_tensor_ms=t_tensor_ms, t_hbm_ms=t_hbm_ms, step_frac=max(t_tensor_ms, t_hbm_ms) / ms_per_step)


def measure_producer(dev, peaks, T=64 * 512, Dm=5120, Hq=40, d=128, steps=10):
    """kara_window_queries (Q projection + RoPE into the window_q layout) for one layer of 64 windows of 512
    tokens at the Qwen3-14B shape; a GEMM, so its roofline is the bf16 tensor peak."""
    import torch
    from paper_2607_01237_b200 import kara
    hid = torch.randn(T, Dm, device=dev).to(torch.bfloat16)
    wq = (torch.randn(Hq * d, Dm, device=dev) / Dm ** 0.5).to(torch.bfloat16)
    pos = (torch.arange(T, device=dev, dtype=torch.int32) % 512) + 20000
    out = torch.empty(T, Hq, d, dtype=torch.bfloat16, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ms = []
    for it in range(3 + steps):
        flush.zero_()
        ev0.record()
        kara.kara_window_queries(hid, wq, pos, 1e6, Hq, d, out=out, max_position=32768)
        ev1.record()
        torch.cuda.synchronize()
        if it >= 3:
            ms.append(ev0.elapsed_time(ev1))
    t = sum(ms) / len(ms)
    tf = 2.0 * T * Dm * Hq * d / (t * 1e-3) / 1e12
    return {"workload": f"SURVEY 8(f)-4 window-query producer: {T} tokens x d_model {Dm} -> {Hq} heads x {d}, RoPE fused",
            "steps": steps, "ms_per_step": t, "tflops": tf, "roofline_frac": tf / peaks["bf16_tflops"], "bound": "tensor",
            "window_queries_per_s": T / (t * 1e-3)}


# -------------------------------------------------------------------------------------------------
def run_gpu(args):
    import torch
    from paper_2607_01237_b200 import kara
    from paper_2607_01237_b200 import replicas

    rank, local_rank, world = replicas.rank_env()
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    replicas.require_devices(world if world > 1 else 1, torch.cuda.device_count())
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    torch.cuda.set_device(local_rank)
    dev = torch.device(f"cuda:{local_rank}")
    kara.lib()
    peaks = _peaks()
    if args.producer_only:
        print(json.dumps({"window_q_producer": measure_producer(dev, peaks, steps=max(args.steps, 1))}))
        return
    variant = "qbuf_only" if args.qbuf_only else "alpha0" if args.alpha0 else "full"

    res = measure(args.workload, args.layers, args.steps, args.warmup, dev, rank, dist, local_rank, simt=args.simt,
                  qbuf_only=args.qbuf_only, alpha0=args.alpha0, score_timing=not args.no_score_timing, want_e2e=True,
                  also_without_events=not args.no_score_timing, want_chain=True)
    e2e_mean = res["e2e"]["mean_s"] if res["e2e"] else 0.0
    total_ms, e2e_mean = replicas.max_over_ranks([res["total_ms"], e2e_mean], dist, dev)
    shape, L, alg = res["shape"], res["L"], res["alg"]
    d = derived(res, peaks, world, total_ms, args.steps)

    if args.qbuf_only:
        # "w/o Bi-Attention": U x n logits per head — 16 x fewer FLOPs at the same K bytes: HBM-bound
        roofline = {"kernel": "score (a1), buffer queries only", "bound": "hbm", "achieved": d["score_gbs"],
                    "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": d["score_gbs"] / peaks["hbm_gbs"] if d["score_gbs"] else None,
                    "bytes_per_launch": alg["score_bytes"]}
    else:
        roofline = {"kernel": "score (a1)", "bound": "tensor", "achieved": d["score_tflops"],
                    "peak": peaks["bf16_tflops"], "unit": "TFLOP/s",
                    "frac": d["score_tflops"] / peaks["bf16_tflops"] if d["score_tflops"] else None,
                    "flops_per_launch": alg["flops"]}
    stale = score_kernel_sha256() != SCORE_KERNEL_SHA256_AT_CAPTURE
    roofline.update({"traffic": None if stale else NCU_SCORE_TRAFFIC_BYTES.get((args.workload, L, variant)),
                     "traffic_source": NCU_TRAFFIC_SOURCE, "traffic_capture_commit": NCU_TRAFFIC_COMMIT,
                     "traffic_stale": stale, "peak_source": peaks["source"] + ", burst",
                     "kernel_ms": d["score_ms"], "share_of_step": d["score_ms"] / d["ms_per_step"]})
    line = {
        "metric": METRIC, "value": d["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": d["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": _config(args.workload, shape, L, {"score_kernel": {1: "simt", 2: "tcgen05+tma"}.get(res["score_path"]),
                                                     "variant": variant, "freed_blocks_per_step": res["freed"]}),
        "kv_gbs": d["kv_gbs"], "algorithmic_gbs": d["algorithmic_gbs"], "step_tflops": d["step_tflops"],
        "clocks": res["clocks"],
        "e2e": ({"value": world * res["wc_step"] / e2e_mean, "unit": UNIT, "h2d_bytes_per_step": res["e2e"]["h2d"],
                 "d2h_bytes_per_step": res["e2e"]["d2h"], "ms_per_step": e2e_mean * 1e3,
                 "api": "kara_compress_window_host (pinned host window_q/tables in, tables + free count out)"}
                if res["e2e"] else None),
        # the same metric for the chain a serving engine runs on the device at a compression event: hidden states (resident)
        # -> kara_window_queries_static (Q projection + RoPE) -> kara_compress_window, layer by layer; rank 0's mean
        "e2e_device_chain": ({"value": res["wc_step"] / (res["chain"]["ms"] * 1e-3), "unit": UNIT,
                              "ms_per_step": res["chain"]["ms"], "producer_ms": res["chain"]["producer_ms"],
                              "compress_ms": res["chain"]["ms"] - res["chain"]["producer_ms"],
                              "producer_tflops": res["chain"]["producer_flops"] / (res["chain"]["producer_ms"] * 1e-3) / 1e12,
                              "steps": res["chain"]["steps"], "d_model": res["chain"]["d_model"],
                              "window_tokens_per_layer": res["chain"]["tokens"],
                              "hidden_bytes_resident": res["chain"]["hidden_bytes"], "h2d_bytes_per_step": 0,
                              "gpu_launches_per_step": res["chain"]["launches"],
                              "api": "per layer: kara_window_queries_static(hidden, W_q[l]) -> window_q[l]; "
                                     "kara_compress_window(l, l+1), KARA_COMMIT on the last; synthetic hidden states"}
                             if res["chain"] else None),
        "gpu_launches": res["launches"],
        # the same step with the library's two event records around the score launch switched off (they sit between the
        # score kernel and the select kernel that is launched programmatically behind it); rank 0's mean, same protocol
        "ms_per_step_no_score_events": res["ms_no_events"],
        "roofline": roofline,
        "step_roofline": {"t_tensor_ms": d["t_tensor_ms"], "t_hbm_ms": d["t_hbm_ms"], "frac": d["step_frac"],
                          "def": "slower of (algorithmic bytes / measured HBM GB/s) and (score FLOPs / measured bf16 TFLOP/s) over ms_per_step"},
    }
    if rank == 0 and world == 1 and not args.no_per_config:
        # the other configs of BASELINE.json (and the prefill workload), a few steps each, same protocol
        per = {}
        for name in ("cfg2", "cfg3", "cfg5", "prefill"):
            if name == args.workload:
                continue
            r = measure(name, 0, 5, 3, dev, rank, None, local_rank)
            dd = derived(r, peaks, 1, None, 5)
            per[name] = {"workload": _workload_label(name, r["shape"]), "n_layers": r["L"], "steps": 5,
                         "ms_per_step": dd["ms_per_step"], "value": dd["value"], "kv_gbs": dd["kv_gbs"],
                         "roofline_frac": dd["score_tflops"] / peaks["bf16_tflops"], "score_kernel_ms": dd["score_ms"],
                         "step_roofline_frac": dd["step_frac"], "freed_blocks_per_step": r["freed"],
                         "gpu_launches": r["launches"], "sm_mhz": r["clocks"]["sm_mhz"]}
        # BASELINE.json configs[3]: retention swept over 10 / 20 / 30 % with the freed-block counts (SURVEY 8(d) expects
        # about 55.75 / 49.56 / 43.38 freed blocks per sequence); the headline above is the 20 % point
        for pct in (10, 30):
            if args.workload != "cfg4":
                break
            r = measure("cfg4", 0, 5, 3, dev, rank, None, local_rank, ratio=pct / 100)
            dd = derived(r, peaks, 1, None, 5)
            per[f"cfg4_r{pct}"] = {"workload": _workload_label("cfg4", r["shape"]) + f", retention {pct} %",
                                   "n_layers": r["L"], "steps": 5, "ms_per_step": dd["ms_per_step"], "value": dd["value"],
                                   "roofline_frac": dd["score_tflops"] / peaks["bf16_tflops"],
                                   "score_kernel_ms": dd["score_ms"], "step_roofline_frac": dd["step_frac"],
                                   "freed_blocks_per_step": r["freed"],
                                   "freed_blocks_per_sequence": r["freed"] / r["shape"].n_seqs,
                                   "gpu_launches": r["launches"], "sm_mhz": r["clocks"]["sm_mhz"]}
        # SURVEY 8(d) timing protocol: cfg 2 also as one call PER LAYER (8 units per call: the latency case of Alg. 1
        # l.6-12) beside the one all-layer call above
        r = measure("cfg2", 0, 5, 3, dev, rank, None, local_rank, per_layer_calls=True, score_timing=False)
        per["cfg2_per_layer_calls"] = {"workload": _workload_label("cfg2", r["shape"]) + ", one call per layer",
                                       "n_layers": r["L"], "calls_per_step": r["L"], "steps": 5,
                                       "ms_per_step": r["total_ms"] / 5, "us_per_call": 1e3 * r["total_ms"] / 5 / r["L"],
                                       "value": r["wc_step"] / (r["total_ms"] / 5 * 1e-3),
                                       "freed_blocks_per_step": r["freed"], "gpu_launches": r["launches"],
                                       "sm_mhz": r["clocks"]["sm_mhz"]}
        per["window_q_producer"] = measure_producer(dev, peaks)
        line["per_config"] = per
    if rank == 0:
        if not args.no_cpu_baseline and world == 1:
            Ls = ORACLE_LAYERS[args.workload]
            small, H, desc = oracle_prepare(shape, Ls, seed=2)
            secs = oracle_leg(small, H, Ls)
            line["cpu_baseline"] = {"value": Ls * small.n_windows / secs, "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": desc, "seconds": secs}
            cores, v_all, wall = oracle_all_cores(args.workload, ORACLE_LAYERS_PER_PROC[args.workload])
            line["cpu_baseline"]["all_cores"] = {
                "value": v_all, "unit": UNIT, "cores": cores, "seconds": wall,
                "how": f"{cores} worker processes (one per core of sched_getaffinity), each the single-threaded oracle on "
                       f"{ORACLE_LAYERS_PER_PROC[args.workload]} layer(s) of its own sequence, started together"}
        print(json.dumps(line))
    if dist:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=list(WORKLOADS))
    ap.add_argument("--layers", type=int, default=0, help="resident layers (default: all that fit)")
    ap.add_argument("--simt", action="store_true", help="force the CUDA-core score kernel")
    ap.add_argument("--qbuf-only", action="store_true",
                    help="ablation 'w/o Bi-Attention' (PAPER.md:L193): score with the buffer's queries only (HBM-bound)")
    ap.add_argument("--alpha0", action="store_true", help="ablation 'w/o Token2Chunk' (PAPER.md:L195): alpha = 0")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config legs (cfg2, cfg3, cfg5, prefill)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--producer-only", action="store_true",
                    help="time only the window-query producer (kara_window_queries) and print its per_config object; "
                         "the command to put under ncu for qproj_kernel")
    ap.add_argument("--no-score-timing", action="store_true",
                    help="no CUDA events inside the library around the score launch (roofline.kernel_ms = 0)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    from paper_2607_01237_b200 import replicas
    if args.impl == "reference":
        run_reference(args)
    elif replicas.needs_spawn(args.gpus):
        # started plainly with --gpus N: start the N ranks (one replica per GPU) and let rank 0 print the line
        import torch
        replicas.require_devices(args.gpus, torch.cuda.device_count())
        sys.exit(replicas.spawn_ranks(args.gpus, [str(Path(__file__).resolve()), *sys.argv[1:]]))
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
