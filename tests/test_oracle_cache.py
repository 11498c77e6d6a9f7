"""Pins for the oracle's O10-O11 and the whole paged path (Eq. 9, Alg. 1 l.11-12, App. C.4;
PAPER.md:L142, L150, L336-337, L354) — CPU only.

Pinned by: numpy fancy indexing (Eq. 9 is a gather by definition), the r=1/alpha=0 no-op, the
closed-form freed-block count, block-conservation (free list U live blocks = all blocks,
disjoint), history bytes untouched, and the synthetic recipe's planted keys surfacing at the top.
"""
import math

import numpy as np
import pytest
import torch

from conftest import torch_bf16_to_bits
from paper_2607_01237_b200 import inputs as kin


def _layout(oracle, wl):
    L, NB, Hkv, bs, d = wl.k_pool.shape
    return oracle.Layout(block_size=bs, n_layers=L, n_kv_heads=Hkv, head_dim=d,
                         sL=NB * Hkv * bs * d, sB=Hkv * bs * d, sH=bs * d, sS=d, num_blocks=NB)


def _host(wl):
    return dict(k=torch_bf16_to_bits(wl.k_pool), v=torch_bf16_to_bits(wl.v_pool),
                q=torch_bf16_to_bits(wl.window_q), bt=wl.block_table.numpy().copy(),
                sl=wl.seq_lens.numpy().copy(), ws=wl.win_start.numpy().copy(),
                fl=wl.free_list.numpy().copy(), fc=wl.free_count.numpy().copy())


def _logical(pool_bits, layer, bt_row, length, head, bs):
    pos = np.arange(length)
    return pool_bits[layer, bt_row[pos // bs], head, pos % bs, :]


# ------------------------------------------------------------------------------------------
def test_compact_rows_is_a_gather(oracle):
    rng = np.random.default_rng(0)
    h, W, U, t, d = 37, 32, 8, 5, 16
    n = W - U
    old = rng.integers(0, 65536, size=(h + W + t, d)).astype(np.uint16)
    F = np.sort(rng.permutation(n)[:9]).astype(np.int32)
    new = oracle.compact_rows(old, h, W, U, t, F)
    expect = np.concatenate([old[:h], old[h + F], old[h + n:]])
    np.testing.assert_array_equal(new, expect)


def test_full_retention_is_a_noop(oracle):
    """r = 1, alpha = 0 => F = [0..n) => nothing moves, nothing freed (SURVEY §8c O10 pin)."""
    shape = kin.scaled(kin.CFG1, ratio=1.0, alpha=0, gamma=3, hist_lo=40, hist_hi=40, tail_hi=3)
    wl = kin.generate(shape, seed=5)
    H = _host(wl)
    k0, v0, bt0, sl0, fc0 = H["k"].copy(), H["v"].copy(), H["bt"].copy(), H["sl"].copy(), H["fc"].copy()
    out = oracle.compress_window(_layout(oracle, wl), H["k"], H["v"], 0, 1, H["bt"], H["sl"], H["ws"],
                                 H["q"], shape.n_q_heads, shape.W, shape.U, shape.ratio, shape.alpha,
                                 shape.gamma, True, H["fl"], H["fc"])
    assert out["keep"] == shape.n
    np.testing.assert_array_equal(out["idx_final"][0, 0, 0], np.arange(shape.n))
    np.testing.assert_array_equal(H["k"], k0)
    np.testing.assert_array_equal(H["v"], v0)
    np.testing.assert_array_equal(H["bt"], bt0)
    np.testing.assert_array_equal(H["sl"], sl0)
    np.testing.assert_array_equal(H["fc"], fc0)


@pytest.mark.parametrize("bs,h,W,U,t,keep", [(16, 256, 64, 8, 0, 12), (16, 4096, 512, 32, 0, 96),
                                             (16, 4099, 512, 32, 7, 96), (256, 1000, 768, 32, 100, 225),
                                             (16, 5, 64, 0, 0, 13), (32, 31, 64, 8, 1, 56)])
def test_metadata_closed_form(oracle, bs, h, W, U, t, keep):
    old_nb = math.ceil((h + W + t) / bs)
    new_nb = math.ceil((h + keep + U + t) / bs)
    NB = old_nb + 9
    rng = np.random.default_rng(h)
    perm = rng.permutation(NB).astype(np.int32)
    bt = np.full((1, old_nb + 2), -1, np.int32)
    bt[0, :old_nb] = perm[:old_nb]
    fl = np.full(NB, -1, np.int32)
    fl[:NB - old_nb] = perm[old_nb:]
    fc = np.array([NB - old_nb], np.int32)
    sl = np.array([h + W + t], np.int32)
    ws = np.array([h], np.int32)
    bt0 = bt.copy()
    oracle.metadata(bt, sl, ws, bs, W, U, keep, fl, fc)
    assert sl[0] == h + keep + U + t
    assert fc[0] - (NB - old_nb) == old_nb - new_nb                      # closed form
    np.testing.assert_array_equal(bt[0, :new_nb], bt0[0, :new_nb])       # prefix unchanged
    assert (bt[0, new_nb:] == -1).all()
    np.testing.assert_array_equal(fl[NB - old_nb:fc[0]], bt0[0, new_nb:old_nb])   # table order
    live = bt[0, :new_nb]
    allb = np.concatenate([live, fl[:fc[0]]])
    assert sorted(allb.tolist()) == list(range(NB))                      # conservation, disjoint


def test_metadata_batch_order(oracle):
    """Reading G16: freed blocks are appended sequence by sequence, each in table order."""
    bs, W, U, keep = 16, 64, 8, 12
    hs = [256, 100, 33]
    nbs = [math.ceil((h + W) / bs) for h in hs]
    NB = sum(nbs)
    bt = np.full((3, max(nbs)), -1, np.int32)
    ids = np.arange(NB, dtype=np.int32)[::-1].copy()
    off = 0
    for s, nb in enumerate(nbs):
        bt[s, :nb] = ids[off:off + nb]
        off += nb
    bt0 = bt.copy()
    fl = np.full(NB, -1, np.int32)
    fc = np.zeros(1, np.int32)
    sl = np.array([h + W for h in hs], np.int32)
    oracle.metadata(bt, sl, np.array(hs, np.int32), bs, W, U, keep, fl, fc)
    expect = []
    for s, h in enumerate(hs):
        expect += bt0[s, math.ceil((h + keep + U) / bs):nbs[s]].tolist()
    assert fl[:fc[0]].tolist() == expect


# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed,tail", [(1, 0), (2, 5), (3, 15)])
def test_whole_path_on_paged_pool(oracle, seed, tail):
    """O1-O11 through the block table equals the per-unit steps applied to the logical rows;
    history bytes and every block not owned by the window are untouched."""
    shape = kin.scaled(kin.CFG1, n_seqs=3, n_layers=2, n_q_heads=4, n_kv_heads=2, hist_lo=19,
                       hist_hi=90, tail_lo=tail, tail_hi=tail)
    wl = kin.generate(shape, seed=seed)
    H = _host(wl)
    k0, v0, bt0, sl0 = H["k"].copy(), H["v"].copy(), H["bt"].copy(), H["sl"].copy()
    fc0 = int(H["fc"][0])
    lay = _layout(oracle, wl)
    out = oracle.compress_window(lay, H["k"], H["v"], 0, 2, H["bt"], H["sl"], H["ws"], H["q"],
                                 shape.n_q_heads, shape.W, shape.U, shape.ratio, shape.alpha,
                                 shape.gamma, True, H["fl"], H["fc"])
    keep, bs, G, n, d = out["keep"], shape.block_size, shape.G, shape.n, shape.head_dim
    assert keep == 12
    freed_total = 0
    for s in range(shape.n_seqs):
        h, old_len = int(H["ws"][s]), int(sl0[s])
        t = old_len - h - shape.W
        new_len = h + keep + shape.U + t
        assert H["sl"][s] == new_len
        freed_total += math.ceil(old_len / bs) - math.ceil(new_len / bs)
        for l in range(2):
            for hk in range(shape.n_kv_heads):
                kold = _logical(k0, l, bt0[s], old_len, hk, bs)
                vold = _logical(v0, l, bt0[s], old_len, hk, bs)
                q = np.ascontiguousarray(H["q"][l, s][:, hk * G:(hk + 1) * G])
                _, A32 = oracle.scores(q, np.ascontiguousarray(kold[h:h + n]))
                np.testing.assert_array_equal(out["scores"][l, s, hk], A32)
                F = oracle.select(A32, keep, shape.alpha, shape.gamma)["F"]
                np.testing.assert_array_equal(out["idx_final"][l, s, hk], F)
                # new logical rows read through the (prefix of the) same block table
                knew = _logical(H["k"], l, bt0[s], new_len, hk, bs)
                vnew = _logical(H["v"], l, bt0[s], new_len, hk, bs)
                np.testing.assert_array_equal(knew, np.concatenate([kold[:h], kold[h + F], kold[h + n:]]))
                np.testing.assert_array_equal(vnew, np.concatenate([vold[:h], vold[h + F], vold[h + n:]]))
    assert int(H["fc"][0]) - fc0 == freed_total
    # blocks that hold no rewritten row are byte-identical (history blocks, other sequences'
    # blocks, free blocks): only blocks covering [h, old_len) of some sequence may differ
    touched = np.zeros(wl.num_blocks, bool)
    for s in range(shape.n_seqs):
        h, old_len = int(H["ws"][s]), int(sl0[s])
        touched[bt0[s, h // bs: math.ceil(old_len / bs)]] = True
    np.testing.assert_array_equal(H["k"][:, ~touched], k0[:, ~touched])
    np.testing.assert_array_equal(H["v"][:, ~touched], v0[:, ~touched])
    # conservation
    live = np.concatenate([H["bt"][s][H["bt"][s] >= 0] for s in range(shape.n_seqs)])
    allb = np.concatenate([live, H["fl"][:H["fc"][0]]])
    assert sorted(allb.tolist()) == list(range(wl.num_blocks))


def test_scores_injected_mode_skips_scoring(oracle):
    shape = kin.scaled(kin.CFG1, n_seqs=2, hist_lo=20, hist_hi=50)
    wl = kin.generate(shape, seed=9)
    H1, H2 = _host(wl), _host(wl)
    lay = _layout(oracle, wl)
    args = (shape.n_q_heads, shape.W, shape.U, shape.ratio, shape.alpha, shape.gamma, True)
    o1 = oracle.compress_window(lay, H1["k"], H1["v"], 0, 1, H1["bt"], H1["sl"], H1["ws"], H1["q"],
                                *args, H1["fl"], H1["fc"])
    o2 = oracle.compress_window(lay, H2["k"], H2["v"], 0, 1, H2["bt"], H2["sl"], H2["ws"], None,
                                *args, H2["fl"], H2["fc"], scores_in=o1["scores"])
    for key in ("k", "v", "bt", "sl", "fl", "fc"):
        np.testing.assert_array_equal(H1[key], H2[key])
    np.testing.assert_array_equal(o1["idx_final"], o2["idx_final"])


# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(1, 9))
def test_cfg1_planted_keys_rank_first(oracle, seed):
    """BASELINE.json configs[0]: 4 planted salient positions (cosine ~0.8 to the mean window
    query) make the top-k unambiguous: they hold ranks 1-4 with a relative margin > 1e-3."""
    wl = kin.generate(kin.CFG1, seed=seed)
    sh = wl.shape
    bt = wl.block_table[0].numpy()
    h = int(wl.win_start[0])
    krows = _logical(torch_bf16_to_bits(wl.k_pool), 0, bt, h + sh.W, 0, sh.block_size)
    q = torch_bf16_to_bits(wl.window_q)[0, 0]
    A64, A32 = oracle.scores(np.ascontiguousarray(q), np.ascontiguousarray(krows[h:h + sh.n]))
    planted = np.flatnonzero(wl.salient[0].numpy())
    assert len(planted) == 4
    order = np.argsort(-A64)
    assert set(order[:4].tolist()) == set(planted.tolist())
    assert A64[order[3]] > A64[order[4]] * (1 + 1e-3)
    out = oracle.select(A32, oracle.budget(sh.n, sh.ratio), sh.alpha, sh.gamma)
    assert set(planted.tolist()) <= set(out["I"].tolist())


def test_generator_is_deterministic_and_conserves_blocks():
    a = kin.generate(kin.scaled(kin.CFG1, n_seqs=4, hist_hi=400), seed=3)
    b = kin.generate(kin.scaled(kin.CFG1, n_seqs=4, hist_hi=400), seed=3)
    assert torch.equal(a.k_pool, b.k_pool) and torch.equal(a.window_q, b.window_q)
    assert torch.equal(a.block_table, b.block_table)
    live = a.block_table[a.block_table >= 0]
    allb = torch.cat([live, a.free_list[: int(a.free_count)]])
    assert sorted(allb.tolist()) == list(range(a.num_blocks))
    assert a.num_blocks >= math.ceil(1.2 * len(live)) - 1
