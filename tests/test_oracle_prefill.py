"""Pins of the oracle's prefill / multi-window function kara_oracle_compress_windows (App. C.2, PAPER.md:L307,
L346; reading G17 in DESIGN.md) against things other than itself:

  * NW windows in one call == NW successive committed single-window calls of kara_oracle_compress_window
    (window w at win_start = h + w (keep + U)): same logical K/V rows, lengths, per-window scores / I / F and the
    same SET of freed blocks (the order differs legitimately: one release at the end vs one per call);
  * numpy fancy-index gather of the definition  new = old[0:h] || (old[h + w W + F_w], buffer_w)_w || tail;
  * NW = 1 is bit-for-bit kara_oracle_compress_window, free-list order included;
  * closed-form length and freed-block count.
"""
import math

import numpy as np
import pytest

from paper_2607_01237_b200 import inputs as kin


@pytest.fixture(scope="module")
def chk(oracle):
    from oracle import check
    return check


def _logical(pool, bt_row, length, layer, head, bs):
    pos = np.arange(length)
    return pool[layer, bt_row[pos // bs], head, pos % bs, :]


SHAPES = [kin.scaled(kin.CFG1, n_windows=3, n_seqs=2, n_layers=2, hist_lo=5, hist_hi=70, tail_lo=0, tail_hi=9),
          kin.scaled(kin.CFG1, n_windows=4, n_seqs=1, hist_lo=0, hist_hi=0),
          kin.scaled(kin.CFG1, n_windows=2, n_seqs=3, n_kv_heads=2, n_q_heads=4, block_size=32, hist_lo=0, hist_hi=40,
                     tail_lo=3, tail_hi=3)]


@pytest.mark.parametrize("shape", SHAPES, ids=lambda s: f"NW{s.n_windows}_S{s.n_seqs}_bs{s.block_size}")
def test_windows_in_one_call_equal_successive_single_window_calls(chk, shape):
    wl = kin.generate(shape, seed=17)
    sh, NW, bs = wl.shape, wl.shape.n_windows, wl.shape.block_size
    L = wl.n_layers_resident
    H0 = chk.host_image(wl)
    A = {k: v.copy() for k, v in H0.items()}
    one = chk.run_oracle(A, sh.n_q_heads, sh.W, sh.U, sh.ratio, sh.alpha, sh.gamma, 0, L, True, n_windows=NW)
    keep = one["keep"]
    B = {k: v.copy() for k, v in H0.items()}
    for w in range(NW):
        B["ws"] = (H0["ws"] + w * (keep + sh.U)).astype(np.int32)
        q_w = np.ascontiguousarray(H0["q"][:, :, w * sh.W:(w + 1) * sh.W])
        Bw = dict(B, q=q_w)
        step = chk.run_oracle(Bw, sh.n_q_heads, sh.W, sh.U, sh.ratio, sh.alpha, sh.gamma, 0, L, True)
        np.testing.assert_array_equal(step["idx_final"], one["idx_final"][:, :, w])
        np.testing.assert_array_equal(step["idx_topk"], one["idx_topk"][:, :, w])
        np.testing.assert_array_equal(step["scores"], one["scores"][:, :, w])
    np.testing.assert_array_equal(A["sl"], B["sl"])
    for s in range(sh.n_seqs):
        ln = int(A["sl"][s])
        nb = math.ceil(ln / bs)
        np.testing.assert_array_equal(A["bt"][s, :nb], B["bt"][s, :nb])
        assert (A["bt"][s, nb:] == -1).all() and (B["bt"][s, nb:] == -1).all()
        for l in range(L):
            for hk in range(sh.n_kv_heads):
                for pool in ("k", "v"):
                    np.testing.assert_array_equal(_logical(A[pool], A["bt"][s], ln, l, hk, bs),
                                                  _logical(B[pool], B["bt"][s], ln, l, hk, bs))
    assert A["fc"][0] == B["fc"][0]
    nf = int(A["fc"][0])
    assert sorted(A["fl"][:nf].tolist()) == sorted(B["fl"][:nf].tolist())


def test_gather_definition_and_closed_forms(chk):
    shape = kin.scaled(kin.CFG1, n_windows=3, n_seqs=2, n_layers=1, hist_lo=11, hist_hi=50, tail_lo=0, tail_hi=7)
    wl = kin.generate(shape, seed=5)
    sh, NW, bs, W, U, n = wl.shape, 3, wl.shape.block_size, wl.shape.W, wl.shape.U, wl.shape.n
    H0 = chk.host_image(wl)
    A = {k: v.copy() for k, v in H0.items()}
    out = chk.run_oracle(A, sh.n_q_heads, W, U, sh.ratio, sh.alpha, sh.gamma, 0, 1, True, n_windows=NW)
    keep = out["keep"]
    freed_total = 0
    for s in range(sh.n_seqs):
        h, ln = int(H0["ws"][s]), int(H0["sl"][s])
        t = ln - h - NW * W
        new_len = h + NW * (keep + U) + t
        assert A["sl"][s] == new_len
        freed_total += math.ceil(ln / bs) - math.ceil(new_len / bs)
        for pool in ("k", "v"):
            old = _logical(H0[pool], H0["bt"][s], ln, 0, 0, bs)
            idx = [np.arange(h)]
            for w in range(NW):
                idx += [h + w * W + out["idx_final"][0, s, w, 0], h + w * W + n + np.arange(U)]
            idx.append(h + NW * W + np.arange(t))
            np.testing.assert_array_equal(_logical(A[pool], A["bt"][s], new_len, 0, 0, bs), old[np.concatenate(idx)])
        # table prefix unchanged, freed entries are the trailing ones in table order
        nb_new, nb_old = math.ceil(new_len / bs), math.ceil(ln / bs)
        np.testing.assert_array_equal(A["bt"][s, :nb_new], H0["bt"][s, :nb_new])
    assert int(A["fc"][0]) - int(H0["fc"][0]) == freed_total
    f0 = int(H0["fc"][0])
    exp = np.concatenate([H0["bt"][s, math.ceil(int(A["sl"][s]) / bs):math.ceil(int(H0["sl"][s]) / bs)]
                          for s in range(sh.n_seqs)])
    np.testing.assert_array_equal(A["fl"][f0:f0 + freed_total], exp)          # batch order, table order (G16)
    # untouched blocks are byte-identical
    touched = set()
    for s in range(sh.n_seqs):
        h, ln = int(H0["ws"][s]), int(H0["sl"][s])
        touched |= set(H0["bt"][s, h // bs:math.ceil(ln / bs)].tolist())
    rest = [b for b in range(wl.num_blocks) if b not in touched]
    np.testing.assert_array_equal(A["k"][:, rest], H0["k"][:, rest])
    np.testing.assert_array_equal(A["v"][:, rest], H0["v"][:, rest])


def test_one_window_is_the_single_window_function(oracle, chk):
    """n_windows = 1 through the C entry point of the prefill function == kara_oracle_compress_window, bit for bit."""
    import ctypes as C
    ko = oracle
    wl = kin.generate(kin.scaled(kin.CFG1, n_seqs=3, hist_lo=10, hist_hi=90, tail_lo=0, tail_hi=6), seed=9)
    sh = wl.shape
    H0 = chk.host_image(wl)
    A = {k: v.copy() for k, v in H0.items()}
    ref = chk.run_oracle(A, sh.n_q_heads, sh.W, sh.U, sh.ratio, sh.alpha, sh.gamma, 0, 1, True)
    B = {k: v.copy() for k, v in H0.items()}
    lay = chk.layout_of(B["k"].shape)
    p = lambda a, ty: a.ctypes.data_as(C.POINTER(ty))
    n, keep = sh.n, ref["keep"]
    sc = np.zeros((1, 3, sh.n_kv_heads, n), np.float32)
    fi = np.zeros((1, 3, sh.n_kv_heads, keep), np.int32)
    rc = ko.lib().kara_oracle_compress_windows(
        C.byref(lay), p(B["k"], C.c_uint16), p(B["v"], C.c_uint16), 0, 1, 3, p(B["bt"], C.c_int32), B["bt"].shape[1],
        p(B["sl"], C.c_int32), p(B["ws"], C.c_int32), 1, p(np.ascontiguousarray(B["q"]), C.c_uint16), sh.n_q_heads,
        sh.W, sh.U, float(sh.ratio), sh.alpha, sh.gamma, 1, p(B["fl"], C.c_int32), p(B["fc"], C.c_int32), None,
        p(sc, C.c_float), None, p(fi, C.c_int32))
    assert rc == 0
    np.testing.assert_array_equal(sc, ref["scores"])
    np.testing.assert_array_equal(fi, ref["idx_final"])
    for key in ("k", "v", "bt", "sl", "fl", "fc"):
        np.testing.assert_array_equal(A[key], B[key])
