"""Parity harness around the CPU oracle — TEST INFRASTRUCTURE ONLY (see kara_oracle.h).

Takes plain numpy images of a workload (and, for the comparison, plain numpy read-backs of what
the CUDA path produced) and runs the three parity stages of DESIGN.md §Parity:

  S1  GPU scores vs oracle O1-O3:  |dA_j| <= 1e-3 * A_j + 1e-6 * (G*W/n)          (all keys)
  S2  oracle O4-O11 re-run on the GPU's own fp32 scores: I, F, every pool byte, block tables,
      seq_lens and the free list must be IDENTICAL
  S3  GPU F vs the oracle's F from its own scores: identical unless one of the unit's decision
      boundaries (k-th/(k+1)-th A, P-th/(P+1)-th R, f-th/(f+1)-th fill candidate) has a relative
      gap < 1e-3 in the oracle ("ambiguous" unit; S2 stands in for it)

Imports nothing from the product package; used by tests/, __graft_entry__.smoke() and bench.py.
"""
from __future__ import annotations

import numpy as np
import torch

from . import kara_oracle as ko

REL_TOL = 1e-3          # north_star: per-key scores within 1e-3 relative, fp32 accumulation
ABS_FLOOR = 1e-6        # x mean score G*W/n (reading G15)


def bits(t: torch.Tensor) -> np.ndarray:
    """bf16 torch tensor (any device) -> uint16 numpy bit patterns."""
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16).copy()


def host_image(wl) -> dict:
    """numpy copies of every array of an inputs.Workload-like object."""
    return dict(k=bits(wl.k_pool), v=bits(wl.v_pool), q=bits(wl.window_q),
                bt=wl.block_table.cpu().numpy().copy(), sl=wl.seq_lens.cpu().numpy().copy(),
                ws=wl.win_start.cpu().numpy().copy(), fl=wl.free_list.cpu().numpy().copy(),
                fc=wl.free_count.cpu().numpy().copy())


def layout_of(k_pool_shape) -> ko.Layout:
    L, NB, Hkv, bs, d = k_pool_shape
    return ko.Layout(block_size=bs, n_layers=L, n_kv_heads=Hkv, head_dim=d, sL=NB * Hkv * bs * d,
                     sB=Hkv * bs * d, sH=bs * d, sS=d, num_blocks=NB)


def run_oracle(H: dict, n_q_heads, W, U, ratio, alpha, gamma, layer_begin, layer_end, commit=True,
               scores_in=None, n_windows=1) -> dict:
    """Runs O1-O11 (or O4-O11 from scores_in) IN PLACE on the numpy image H; returns the dumps."""
    lay = layout_of(H["k"].shape)
    q = None if scores_in is not None else np.ascontiguousarray(H["q"][layer_begin:layer_end])
    return ko.compress_window(lay, H["k"], H["v"], layer_begin, layer_end, H["bt"], H["sl"], H["ws"], q,
                              n_q_heads, W, U, ratio, alpha, gamma, commit, H["fl"], H["fc"],
                              scores_in=scores_in, n_windows=n_windows)


def score_tolerance(A_ref: np.ndarray, G: int, W: int, n: int) -> np.ndarray:
    return REL_TOL * np.abs(A_ref) + ABS_FLOOR * (G * W / n)


def _rel_gap(hi: float, lo: float) -> float:
    return abs(hi - lo) / max(abs(hi), 1e-300)


def is_ambiguous(A32: np.ndarray, keep: int, alpha: int, gamma: int, rel: float = REL_TOL) -> bool:
    """True if any of the unit's three decision boundaries is closer than `rel` (relative)."""
    A = A32.astype(np.float64)
    n = len(A)
    k = keep - alpha
    P = alpha // (gamma - 2)
    order = np.argsort(-A, kind="stable")
    if k < n and _rel_gap(A[order[k - 1]], A[order[k]]) < rel:
        return True
    sel = ko.select(A32, keep, alpha, gamma)
    I = sel["I"]
    a, b = I[:-1], I[1:]
    elig = ((b - a) < gamma) & ((b - a - 1) >= 1)
    R = (np.float32(A32[a] + A32[b]) * (b - a - 1).astype(np.float32)).astype(np.float64)[elig]
    R = np.sort(R)[::-1]
    if 0 < P < len(R) and _rel_gap(R[P - 1], R[P]) < rel:
        return True
    f = keep - k - sel["n_chunk_added"]
    hat = np.zeros(n, bool)
    hat[I] = True
    for t in sel["chunks"]:
        if t >= 0:
            hat[I[t] + 1:I[t + 1]] = True
    rest = np.sort(A[~hat])[::-1]
    if 0 < f < len(rest) and _rel_gap(rest[f - 1], rest[f]) < rel:
        return True
    return False


def compare(H0: dict, gpu: dict, n_q_heads, W, U, ratio, alpha, gamma, layer_begin, layer_end,
            commit=True, check_s1=True, n_windows=1) -> dict:
    """H0: pristine numpy image.  gpu: numpy read-backs of the CUDA path after its call:
    k, v (pool bits), bt, sl, fl, fc, scores [L,S,Hkv,n], idx_topk [..,k], idx_final [..,keep].
    Raises AssertionError on any parity failure; returns statistics."""
    Hkv = H0["k"].shape[2]
    G = n_q_heads // Hkv
    n = W - U
    stats = {}
    # ---- oracle on its own scores (S1, S3) ----
    Ho = {k_: v_.copy() for k_, v_ in H0.items()}
    own = run_oracle(Ho, n_q_heads, W, U, ratio, alpha, gamma, layer_begin, layer_end, commit, n_windows=n_windows)
    keep = own["keep"]
    if n_windows > 1:      # the GPU read-backs are [L, S, NW, Hkv, .] too; fold (S, NW) into one axis for the loops below
        own = {k_: (v_.reshape((v_.shape[0], -1) + v_.shape[3:]) if isinstance(v_, np.ndarray) else v_) for k_, v_ in own.items()}
        gpu = dict(gpu)
        for k_ in ("scores", "idx_topk", "idx_final"):
            gpu[k_] = gpu[k_].reshape((gpu[k_].shape[0], -1) + gpu[k_].shape[3:])
    if check_s1:
        err = np.abs(gpu["scores"].astype(np.float64) - own["scores"].astype(np.float64))
        tol = score_tolerance(own["scores"].astype(np.float64), G, W, n)
        worst = float((err / tol).max())
        stats["s1_worst_err_over_tol"] = worst
        stats["s1_max_rel_err"] = float((err / np.maximum(np.abs(own["scores"]), 1e-30)).max())
        assert worst <= 1.0, f"S1: score error {worst:.3f} x tolerance"
    # ---- S2: oracle from the GPU's scores must reproduce everything bit for bit ----
    Hs = {k_: v_.copy() for k_, v_ in H0.items()}
    inj = run_oracle(Hs, n_q_heads, W, U, ratio, alpha, gamma, layer_begin, layer_end, commit,
                     scores_in=np.ascontiguousarray(gpu["scores"], np.float32), n_windows=n_windows)
    if n_windows > 1:
        inj = {k_: (v_.reshape((v_.shape[0], -1) + v_.shape[3:]) if isinstance(v_, np.ndarray) else v_) for k_, v_ in inj.items()}
    np.testing.assert_array_equal(gpu["idx_topk"], inj["idx_topk"], err_msg="S2: I differs")
    np.testing.assert_array_equal(gpu["idx_final"], inj["idx_final"], err_msg="S2: F differs")
    np.testing.assert_array_equal(gpu["k"], Hs["k"], err_msg="S2: K pool bytes differ")
    np.testing.assert_array_equal(gpu["v"], Hs["v"], err_msg="S2: V pool bytes differ")
    np.testing.assert_array_equal(gpu["bt"], Hs["bt"], err_msg="S2: block tables differ")
    np.testing.assert_array_equal(gpu["sl"], Hs["sl"], err_msg="S2: seq_lens differ")
    np.testing.assert_array_equal(gpu["fc"], Hs["fc"], err_msg="S2: free_count differs")
    nfree = int(Hs["fc"][0])
    np.testing.assert_array_equal(gpu["fl"][:nfree], Hs["fl"][:nfree], err_msg="S2: free list differs")
    # ---- S3: end-to-end index sets ----
    units = amb = mism = 0
    Ls, S = own["idx_final"].shape[:2]
    for l in range(Ls):
        for s in range(S):
            for hk in range(Hkv):
                units += 1
                same = np.array_equal(gpu["idx_final"][l, s, hk], own["idx_final"][l, s, hk])
                if not same:
                    if is_ambiguous(own["scores"][l, s, hk], keep, alpha, gamma):
                        amb += 1
                    else:
                        mism += 1
    stats.update(units=units, s3_ambiguous_mismatch=amb, s3_hard_mismatch=mism, keep=keep)
    assert mism == 0, f"S3: {mism} of {units} units differ from the oracle with no near-tie to excuse it"
    return stats
