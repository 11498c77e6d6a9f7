"""Seeded synthetic workloads for Kara's compress_window step (inputs only).

This module is the ONE thing the CUDA path's tests/bench and the CPU oracle's tests share.  It
holds none of the method's arithmetic (no scoring, selection, Token2Chunk or compaction): it
draws K/V/Q values, lays logical rows into a paged pool through a random block table, and
builds the free list.  It imports neither the CUDA binding nor the oracle.

The recipes follow BASELINE.json `configs` with the hyper-parameters SURVEY.md §8(d) fixes from
the paper (gamma=8, alpha=32, U=32: PAPER.md:L275, L285) and are restated in DESIGN.md §Inputs.
They stand in for the paper's serving workload (R1-Llama-8B / Qwen3 on MATH-500),
which is not available here: same shapes (Qwen3-14B-like GQA 40/8 x 128), window lengths and
retention; values are synthetic.

Physical layout written here (the product's layout, include/kara.h):
    k_pool, v_pool : bf16 [n_layers][num_blocks][n_kv_heads][block_size][head_dim]
    logical token p of sequence s lives in block block_table[s][p // block_size], slot p % block_size.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import torch


@dataclass(frozen=True)
class KaraShape:
    """One named workload.  Lengths in tokens."""
    name: str
    n_seqs: int
    n_layers: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    block_size: int
    W: int                       # window length |W|
    U: int                       # protected buffer |U| at the window's end
    ratio: float                 # retention r of the compressible region
    alpha: int                   # Token2Chunk budget
    gamma: int                   # max chunk length incl. endpoints
    hist_lo: int                 # history length h ~ U{hist_lo..hist_hi} per sequence
    hist_hi: int
    tail_lo: int = 0             # tail t ~ U{tail_lo..tail_hi} tokens after the window (App. C.4)
    tail_hi: int = 0
    q_shift: float = 2.0         # shared query-mean component c * v_hat (SURVEY §8d note)
    k_dist: str = "normal"       # "normal" | "student_t3"
    n_outlier_channels: int = 4  # key channels scaled x5
    outlier_scale: float = 5.0
    planted_positions: int = 0   # cfg 1: this many isolated salient positions
    salient_frac: float = 0.0    # cfg 2+: fraction of window positions in salient runs
    run_lo: int = 2
    run_hi: int = 16
    pool_slack: float = 1.2      # num_blocks = ceil(slack * live blocks)
    n_windows: int = 1           # prefill (App. C.2): this many disjoint windows of W tokens per sequence

    @property
    def n(self) -> int:
        return self.W - self.U

    @property
    def G(self) -> int:
        return self.n_q_heads // self.n_kv_heads


# BASELINE.json configs[0..4] (1-based "cfg N" in SURVEY.md / DESIGN.md).
CFG1 = KaraShape("cfg1_tiny", 1, 1, 4, 1, 64, 16, W=64, U=8, ratio=0.2, alpha=4, gamma=4,
                 hist_lo=256, hist_hi=256, n_outlier_channels=0, planted_positions=4)
CFG2 = KaraShape("cfg2_qwen3_14b_1seq", 1, 40, 40, 8, 128, 16, W=512, U=32, ratio=0.2, alpha=32,
                 gamma=8, hist_lo=4096, hist_hi=4096, salient_frac=0.05)
CFG3 = KaraShape("cfg3_batch64", 64, 40, 40, 8, 128, 16, W=512, U=32, ratio=0.2, alpha=32, gamma=8,
                 hist_lo=2048, hist_hi=16384, salient_frac=0.05)
CFG4 = KaraShape("cfg4_serving256", 256, 40, 40, 8, 128, 16, W=1024, U=32, ratio=0.2, alpha=32,
                 gamma=8, hist_lo=8192, hist_hi=32768, salient_frac=0.05, pool_slack=1.0 / 0.95)
CFG5 = KaraShape("cfg5_longcot", 16, 64, 64, 8, 128, 16, W=2048, U=64, ratio=0.2, alpha=32, gamma=8,
                 hist_lo=65536, hist_hi=131072, k_dist="student_t3", salient_frac=0.05, run_lo=1,
                 run_hi=64)
# a prompt split into windows of W and compressed in one call: 8 prompts of
# 16 x 512 tokens, no compressed history in front, same attention shape and hyper-parameters as cfg 2/3.
PREFILL = KaraShape("prefill_8x16x512", 8, 40, 40, 8, 128, 16, W=512, U=32, ratio=0.2, alpha=32, gamma=8,
                    hist_lo=0, hist_hi=0, salient_frac=0.05, n_windows=16)
CONFIGS = {c.name: c for c in (CFG1, CFG2, CFG3, CFG4, CFG5, PREFILL)}


def scaled(shape: KaraShape, **kw) -> KaraShape:
    """A reduced copy (fewer layers / sequences / shorter histories) for parity cases."""
    return replace(shape, **kw)


@dataclass
class Workload:
    shape: KaraShape
    seed: int
    n_layers_resident: int
    num_blocks: int
    max_blocks: int
    k_pool: torch.Tensor          # bf16 [L, NB, Hkv, bs, d]
    v_pool: torch.Tensor
    window_q: torch.Tensor        # bf16 [L, S, n_windows * W, Hq, d]
    block_table: torch.Tensor     # int32 [S, max_blocks], -1 padded
    seq_lens: torch.Tensor        # int32 [S]
    win_start: torch.Tensor       # int32 [S]
    free_list: torch.Tensor       # int32 [NB]; first free_count entries valid
    free_count: torch.Tensor      # int32 [1]
    salient: torch.Tensor         # bool [S, n] planted positions (for tests' sanity checks)
    meta: dict = field(default_factory=dict)


def _unit(x: torch.Tensor) -> torch.Tensor:
    return x / x.norm(dim=-1, keepdim=True).clamp_min(1e-20)


def _salient_mask(shape: KaraShape, gen: torch.Generator) -> torch.Tensor:
    """bool [S, n] on CPU: isolated planted positions (cfg 1) or contiguous runs (cfg 2+)."""
    S, n = shape.n_seqs, shape.n
    mask = torch.zeros(S, n, dtype=torch.bool)
    for s in range(S):
        if shape.planted_positions > 0:
            # isolated: no two planted positions adjacent
            perm = torch.randperm(n // 2, generator=gen)[: shape.planted_positions]
            mask[s, perm * 2] = True
        target = int(round(shape.salient_frac * n))
        covered, guard = 0, 0
        while covered < target and guard < 10 * n:
            guard += 1
            ln = int(torch.randint(shape.run_lo, shape.run_hi + 1, (1,), generator=gen))
            ln = min(ln, n)
            st = int(torch.randint(0, n - ln + 1, (1,), generator=gen))
            new = int((~mask[s, st:st + ln]).sum())
            mask[s, st:st + ln] = True
            covered += new
    return mask


def generate(shape: KaraShape, seed: int, device: str | torch.device = "cpu",
             n_layers_resident: int | None = None, history_fill: str = "randn") -> Workload:
    """Draw one workload.  All randomness comes from `seed` (CPU generator for the structure,
    a generator on `device` for the values), so the same (shape, seed, device kind) reproduces
    the same bits.  `history_fill`: "randn" (values like the window's) or "pattern" (cheap
    address pattern; the history is never read by the method, only checked for identity)."""
    dev = torch.device(device)
    L = shape.n_layers if n_layers_resident is None else int(n_layers_resident)
    S, W, U, n = shape.n_seqs, shape.W, shape.U, shape.n
    NW = shape.n_windows
    Hq, Hkv, d, bs, G = shape.n_q_heads, shape.n_kv_heads, shape.head_dim, shape.block_size, shape.G
    cg = torch.Generator(device="cpu").manual_seed(int(seed))
    vg = torch.Generator(device=dev).manual_seed(int(seed) ^ 0x5DEECE66D)

    # ---- structure: lengths, block tables, free list (CPU, exact integers) -------------------
    h = torch.randint(shape.hist_lo, shape.hist_hi + 1, (S,), generator=cg, dtype=torch.int64)
    t = torch.randint(shape.tail_lo, shape.tail_hi + 1, (S,), generator=cg, dtype=torch.int64)
    seq_len = h + NW * W + t
    nblk = (seq_len + bs - 1) // bs
    live = int(nblk.sum())
    num_blocks = max(int(math.ceil(shape.pool_slack * live)), live)
    max_blocks = int(nblk.max())
    perm = torch.randperm(num_blocks, generator=cg).to(torch.int32)
    block_table = torch.full((S, max_blocks), -1, dtype=torch.int32)
    off = 0
    for s in range(S):
        nb = int(nblk[s])
        block_table[s, :nb] = perm[off:off + nb]
        off += nb
    free_list = torch.full((num_blocks,), -1, dtype=torch.int32)
    n_free = num_blocks - live
    free_list[:n_free] = perm[off:]
    free_count = torch.tensor([n_free], dtype=torch.int32)
    salient = _salient_mask(shape, cg)

    # ---- values ------------------------------------------------------------------------------
    k_pool = torch.empty((L, num_blocks, Hkv, bs, d), dtype=torch.bfloat16, device=dev)
    v_pool = torch.empty_like(k_pool)
    window_q = torch.empty((L, S, NW * W, Hq, d), dtype=torch.bfloat16, device=dev)
    out_ch = torch.randperm(d, generator=cg)[: shape.n_outlier_channels].to(dev)
    bt_dev = block_table.to(dev).long()
    sal_dev = salient.to(dev)

    def randn(*sz):
        return torch.randn(*sz, generator=vg, device=dev, dtype=torch.float32)

    def draw_k(*sz):
        x = randn(*sz)
        if shape.k_dist == "student_t3":
            chi = randn(*sz, 3).square().sum(-1) / 3.0
            x = x / chi.sqrt().clamp_min(1e-6)
        elif shape.k_dist != "normal":
            raise ValueError(shape.k_dist)
        if shape.n_outlier_channels:
            x[..., out_ch] *= shape.outlier_scale
        return x

    for l in range(L):
        if history_fill == "pattern":
            pat = torch.arange(num_blocks * Hkv * bs * d, device=dev, dtype=torch.int32)
            pat = ((pat * 40503 + l * 977) & 0x3FFF).to(torch.int16)  # small finite bf16 patterns
            k_pool[l].view(torch.int16).copy_(pat.view(num_blocks, Hkv, bs, d))
            v_pool[l].view(torch.int16).copy_((pat ^ 0x155).view(num_blocks, Hkv, bs, d))
        elif history_fill == "randn":
            k_pool[l].copy_(draw_k(num_blocks, Hkv, bs, d))
            v_pool[l].copy_(randn(num_blocks, Hkv, bs, d))
        else:
            raise ValueError(history_fill)
        for s in range(S):
          for w in range(NW):
            # window queries: N(0,1) + c * v_hat per (layer, seq, window, kv head)
            v_hat = _unit(randn(Hkv, d))
            q = randn(W, Hkv, G, d) + shape.q_shift * v_hat[None, :, None, :]
            q_bf = q.to(torch.bfloat16)
            window_q[l, s, w * W:(w + 1) * W] = q_bf.view(W, Hq, d)
            # window (+ tail behind the last window) keys / values
            wt = W + (int(t[s]) if w == NW - 1 else 0)
            kw = draw_k(wt, Hkv, d)
            vw = randn(wt, Hkv, d)
            if bool(salient[s].any()):
                # planted keys: keep the norm, point 0.8 along the unit mean window query of the
                # unit and 0.6 along the key's own orthogonal remainder (cosine 0.8 recipe)
                u_hat = _unit(q_bf.float().mean(dim=(0, 2)))            # [Hkv, d]
                kc = kw[:n]                                             # [n, Hkv, d]
                nrm = kc.norm(dim=-1, keepdim=True)
                orth = _unit(kc - (kc * u_hat).sum(-1, keepdim=True) * u_hat)
                planted = nrm * (0.8 * u_hat + 0.6 * orth)
                kw[:n] = torch.where(sal_dev[s][:, None, None], planted, kc)
            pos = torch.arange(int(h[s]) + w * W, int(h[s]) + w * W + wt, device=dev)
            blk = bt_dev[s, pos // bs]
            slot = pos % bs
            k_pool[l, blk, :, slot, :] = kw.to(torch.bfloat16)
            v_pool[l, blk, :, slot, :] = vw.to(torch.bfloat16)

    return Workload(shape=shape, seed=int(seed), n_layers_resident=L, num_blocks=num_blocks,
                    max_blocks=max_blocks, k_pool=k_pool, v_pool=v_pool, window_q=window_q,
                    block_table=block_table.to(dev), seq_lens=seq_len.to(torch.int32).to(dev),
                    win_start=h.to(torch.int32).to(dev), free_list=free_list.to(dev),
                    free_count=free_count.to(dev), salient=salient,
                    meta={"live_blocks": live, "tail": t.tolist(), "outlier_channels": out_ch.tolist()})


def logical_rows(pool: torch.Tensor, layer: int, block_table_row: torch.Tensor, length: int,
                 kv_head: int) -> torch.Tensor:
    """Dense [length, d] view of one (layer, sequence, kv head) read through the block table —
    pure indexing of the documented layout (used by tests to look at the pool directly)."""
    bs = pool.shape[3]
    pos = torch.arange(length, device=pool.device)
    blk = block_table_row.long()[pos // bs]
    return pool[layer, blk, kv_head, pos % bs, :]
