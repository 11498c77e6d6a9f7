"""GPU-side helpers of the parity tests: run the CUDA path through the C ABI binding and read
everything back as numpy.  Imports the product only; the comparison lives in oracle/check.py."""
from __future__ import annotations

import numpy as np
import torch

from paper_2607_01237_b200 import kara


def bits(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16).copy()


def to_cuda(wl):
    """Device copies of a CPU workload's tensors (the CPU workload stays pristine)."""
    dev = torch.device("cuda:0")
    return dict(k=wl.k_pool.to(dev), v=wl.v_pool.to(dev), q=wl.window_q.to(dev),
                bt=wl.block_table.to(dev), sl=wl.seq_lens.to(dev), ws=wl.win_start.to(dev),
                fl=wl.free_list.to(dev), fc=wl.free_count.to(dev))


def gpu_compress(wl, layer_begin=None, layer_end=None, flags=kara.KARA_COMMIT | kara.KARA_KEEP_DEBUG,
                 use_win_start=True, dev_tensors=None, overrides=None):
    """Runs kara_compress_window on a copy of workload `wl`; returns (readback dict, cache, D)."""
    sh = wl.shape
    p = dict(W=sh.W, U=sh.U, ratio=sh.ratio, alpha=sh.alpha, gamma=sh.gamma)
    p.update(overrides or {})
    D = dev_tensors or to_cuda(wl)
    L = D["k"].shape[0]
    lb = 0 if layer_begin is None else layer_begin
    le = L if layer_end is None else layer_end
    cache = kara.KaraCache(sh.block_size, L, sh.n_kv_heads, sh.head_dim)
    cache.attach_pool(D["k"], D["v"], D["fl"], D["fc"])
    NW = getattr(sh, "n_windows", 1)
    if NW > 1:      # prefill: kara_compress_windows
        cache.compress_windows(lb, le, D["bt"], D["sl"], D["ws"] if use_win_start else None, NW,
                               D["q"][lb:le].contiguous(), p["W"], p["U"], p["ratio"], p["alpha"], p["gamma"], flags)
    else:
        cache.compress_window(lb, le, D["bt"], D["sl"], D["ws"] if use_win_start else None,
                              D["q"][lb:le].contiguous(), p["W"], p["U"], p["ratio"], p["alpha"], p["gamma"], flags)
    torch.cuda.synchronize()
    out = readback(cache, D, lb, le, sh.n_seqs, sh.n_kv_heads, flags, n_windows=NW)
    return out, cache, D


def readback(cache, D, lb, le, n_seqs, n_kv_heads, flags, n_windows=1):
    out = dict(k=bits(D["k"]), v=bits(D["v"]), bt=D["bt"].cpu().numpy().copy(), sl=D["sl"].cpu().numpy().copy(),
               fl=D["fl"].cpu().numpy().copy(), fc=D["fc"].cpu().numpy().copy(), status=cache.status())
    if flags & kara.KARA_KEEP_DEBUG:
        sc, it, fi = [], [], []
        for l in range(lb, le):
            for s in range(n_seqs * n_windows):      # after a multi-window call `seq` is sequence * n_windows + window
                for hk in range(n_kv_heads):
                    sc.append(cache.gather_debug(kara.KARA_DBG_SCORES, l, s, hk))
                    it.append(cache.gather_debug(kara.KARA_DBG_IDX_TOPK, l, s, hk))
                    fi.append(cache.gather_debug(kara.KARA_DBG_IDX_FINAL, l, s, hk))
        shp = (le - lb, n_seqs, n_kv_heads, -1) if n_windows == 1 else (le - lb, n_seqs, n_windows, n_kv_heads, -1)
        out.update(scores=np.stack(sc).reshape(shp), idx_topk=np.stack(it).reshape(shp),
                   idx_final=np.stack(fi).reshape(shp))
    return out
