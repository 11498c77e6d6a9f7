"""Per-role clock64 time stamps of the score kernel (CTA 0), for a library built with the trace switch:

    KARA_NVCC_EXTRA=-DKARA_TC_TRACE python -m paper_2607_01237_b200.build --force
    python paper_2607_01237_b200/profiling/score_trace.py [cfg3|cfg4|cfg5]
    python -m paper_2607_01237_b200.build --force            # back to the product build

Workload: 16 sequences of cfg3's shape x 8 layers (clusters of 2; default), or of cfg4's / cfg5's x 2 layers (clusters of 4 / 8).  Columns per role (cycles since tile 8's first MMA wait):
  B0 / B15 (pass-B warps 0 and 15): 0 wait for S half 0 | 1 got it, TMEM load issued | 2 (wait::ld) | 3 piece 0 done, half 1
            load issued | 4 piece 1 done, (z, l) published | 5 arrived on bdone
  MMA: 0 wait for the Q tile | 1 got it | 2 TMEM half 0 free | 3 half 0 issued | 4 half 1 free | 5 half 1 issued
  C16 / C17 (pass-C warps of quadrants 0 and 1): 0 wait for bdone | 1 got it | 2 statistics sent to the peer CTA | 3 peer's
            arrived | 4 weights written | 5 TMEM half 0 read and released | 6 half 1 released
"""
import ctypes as C
import sys
from pathlib import Path

import numpy as np
import torch

sys.path.insert(0, str(Path(__file__).resolve().parents[2]))
from paper_2607_01237_b200 import inputs as kin, kara  # noqa: E402

L = kara.lib()
if not hasattr(L, "kara_tc_trace_read"):
    raise SystemExit("libkara.so was not built with -DKARA_TC_TRACE (see the header of this file)")
base = {"cfg3": kin.CFG3, "cfg4": kin.CFG4, "cfg5": kin.CFG5}[sys.argv[1] if len(sys.argv) > 1 else "cfg3"]
sh = kin.scaled(base, n_seqs=16, n_layers=8 if base is kin.CFG3 else 2, hist_lo=2048, hist_hi=4096)
nL = sh.n_layers
wl = kin.generate(sh, seed=3, device="cuda", n_layers_resident=nL, history_fill="pattern")
cache = kara.KaraCache(sh.block_size, nL, sh.n_kv_heads, sh.head_dim)
cache.attach_pool(wl.k_pool, wl.v_pool, wl.free_list, wl.free_count)
for _ in range(2):
    cache.compress_window(0, nL, wl.block_table, wl.seq_lens, wl.win_start, wl.window_q, sh.W, sh.U, sh.ratio, sh.alpha,
                          sh.gamma, 0)
    torch.cuda.synchronize()
n = 5 * 64 * 8
buf = np.zeros(n, np.int64)
L.kara_tc_trace_read.argtypes = [C.c_void_p, C.c_int]
assert L.kara_tc_trace_read(buf.ctypes.data, n) == 0
t = buf.reshape(5, 64, 8)
t0 = t[2, 8, 0]
names = ["B0", "B15", "MMA", "C16", "C17"]
for ti in range(8, 20):
    for r in range(5):
        print(ti, names[r], " ".join(f"{int(x - t0):7d}" if x else "      -" for x in t[r, ti]))
per = np.diff(t[2, 8:60, 1])
print("cycles per tile (MMA warp, tiles 8..59): mean", per.mean(), "median", np.median(per))
