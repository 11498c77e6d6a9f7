"""Pins of the oracle's periodic compression policy (kara_oracle_policy_step / _commit: PAPER.md Alg. 1, L311-344 as
reconstructed by reading G12; App. C.4; B.1, L275) against things other than itself:

* a TOKEN-LEVEL simulation in plain Python in which every token carries its own "compressed" flag and every block its
  own owner — eligibility is then literally "the W tokens in front of the partial last block are all uncompressed"
  (Alg. 1 l.5 + C.4), with no counter anywhere;
* the paper's KvLLM setting (block 256, W = 768 = 3 blocks, delta = 128): closed-form first compression event;
* hand-worked allocation order, the max_select cap, pool exhaustion, block conservation.
"""
import numpy as np
import pytest


def _pool(n_seqs, max_blocks, num_blocks, rng):
    bt = np.full((n_seqs, max_blocks), -1, np.int32)
    fl = np.full(num_blocks, -1, np.int32)
    fl[:] = rng.permutation(num_blocks).astype(np.int32)
    return bt, fl, np.array([num_blocks], np.int32)


class TokenModel:
    """Independent model: per sequence a list of booleans (token compressed?) and a list of owned blocks."""

    def __init__(self, n_seqs, bs, free_stack):
        self.bs = bs
        self.tok = [[] for _ in range(n_seqs)]
        self.blocks = [[] for _ in range(n_seqs)]
        self.free = list(free_stack)            # top of the stack = end of the list

    def decode(self, s):
        if len(self.tok[s]) % self.bs == 0:
            self.blocks[s].append(self.free.pop())
        self.tok[s].append(False)

    def window(self, s, W):
        """Start of the window of W uncompressed tokens in front of the partial last block, or None."""
        ln = len(self.tok[s])
        end = ln - ln % self.bs
        if end - W < 0 or any(self.tok[s][end - W:end]):
            return None
        return end - W

    def compress(self, s, h, W, U, keep):
        n = W - U
        self.tok[s] = self.tok[s][:h] + [True] * keep + self.tok[s][h + n:]       # retained rows, then buffer + tail
        nb = -(-len(self.tok[s]) // self.bs)
        while len(self.blocks[s]) > nb:                                            # trailing blocks, table order
            self.free.append(self.blocks[s].pop(nb))


@pytest.mark.parametrize("bs,W,U,keep,delta,m,S,steps,seed", [(16, 64, 8, 12, 8, 2, 5, 400, 1), (4, 12, 2, 3, 5, 3, 7, 300, 2),
                                                              (8, 24, 0, 5, 3, 1, 4, 250, 3), (16, 48, 16, 7, 16, 8, 6, 500, 4)])
def test_policy_against_token_level_simulation(oracle, bs, W, U, keep, delta, m, S, steps, seed):
    rng = np.random.default_rng(seed)
    max_blocks, NB = 64, 400
    bt, fl, fc = _pool(S, max_blocks, NB, rng)
    model = TokenModel(S, bs, fl.tolist())
    sl, un, g = np.zeros(S, np.int32), np.zeros(S, np.int32), np.zeros(1, np.int32)
    events = 0
    for step in range(steps):
        active = (rng.random(S) < 0.9).astype(np.uint8)
        sel = oracle.policy_step(bt, sl, un, active, fl, fc, g, bs, delta, W, m)
        for s in range(S):
            if active[s]:
                model.decode(s)
        # expected selection from the token flags alone
        exp = []
        if (step + 1) > W and (step + 1) % delta == 0:
            for s in range(S):
                if active[s] and len(exp) < m:
                    h = model.window(s, W)
                    if h is not None:
                        exp.append((s, h))
        assert sel["sel_count"] == len(exp)
        assert [(int(a), int(b)) for a, b in zip(sel["sel_ids"][:len(exp)], sel["sel_win_start"][:len(exp)])] == exp
        assert np.all(sel["sel_ids"][len(exp):] == -1) and np.all(sel["sel_seq_lens"][len(exp):] == -1)
        if exp:
            events += 1
            n_sel = len(exp)
            # "Kara" on the selected sub-batch: only its metadata matters here (O11, pinned elsewhere)
            oracle.metadata(sel["sel_block_table"][:n_sel], sel["sel_seq_lens"][:n_sel], sel["sel_win_start"][:n_sel], bs, W,
                            U, keep, fl, fc)
            oracle.policy_commit(sel, keep, U, bt, sl, un)
            for s, h in exp:
                model.compress(s, h, W, U, keep)
        # state equals the token-level model after every step
        for s in range(S):
            assert sl[s] == len(model.tok[s])
            trailing = 0
            for f in reversed(model.tok[s]):
                if f:
                    break
                trailing += 1
            assert un[s] == trailing
            nb = len(model.blocks[s])
            assert bt[s, :nb].tolist() == model.blocks[s] and np.all(bt[s, nb:] == -1)
        assert fl[:int(fc[0])].tolist() == model.free
        live = np.concatenate([bt[s][bt[s] >= 0] for s in range(S)])
        assert sorted(np.concatenate([live, fl[:int(fc[0])]]).tolist()) == list(range(NB))      # conservation
    assert events > 0


def test_kvllm_setting_first_event(oracle):
    """PAPER.md B.1 (L271-275): block 256, window = 3 blocks = 768 tokens, delta = 128.  A sequence decoding from an
    empty cache is first selected at the smallest g with g > 768, g mod 128 = 0 and g - (g mod 256) >= 768: g = 896
    (t = 128 tokens in the partial block, window = the three full blocks [0, 768))."""
    bs, W, delta = 256, 768, 128
    bt, fl, fc = _pool(1, 16, 32, np.random.default_rng(0))
    sl, un, g = np.zeros(1, np.int32), np.zeros(1, np.int32), np.zeros(1, np.int32)
    first = None
    for step in range(1, 1200):
        sel = oracle.policy_step(bt, sl, un, None, fl, fc, g, bs, delta, W, 30)
        if sel["sel_count"]:
            first = (step, int(sel["sel_win_start"][0]), int(sel["sel_seq_lens"][0]))
            break
    assert first == (896, 0, 896)
    # "257 KV pairs retained per window" incl. the buffer of 32 (L275): keep + U = 257 -> new length 257 + 128
    keep, U = 225, 32
    oracle.metadata(sel["sel_block_table"][:1], sel["sel_seq_lens"][:1], sel["sel_win_start"][:1], bs, W, U, keep, fl, fc)
    oracle.policy_commit(sel, keep, U, bt, sl, un)
    assert sl[0] == 257 + 128 and un[0] == 32 + 128
    assert int(fc[0]) == 32 - 2                       # 4 blocks held before, ceil(385 / 256) = 2 after
    # the window moves on once W - U new uncompressed tokens exist beyond it (L346): next event needs
    # uncompressed - t >= 768 again
    nxt = None
    for step in range(897, 3000):
        sel = oracle.policy_step(bt, sl, un, None, fl, fc, g, bs, delta, W, 30)
        if sel["sel_count"]:
            nxt = (step, int(sel["sel_win_start"][0]), int(sel["sel_seq_lens"][0]))
            break
    # length after s more steps: 385 + s; uncompressed 160 + s; need (160 + s) - ((385 + s) mod 256) >= 768 at a multiple of 128
    exp = next(st for st in range(897, 3000) if st % 128 == 0 and (160 + st - 896) - ((385 + st - 896) % 256) >= 768)
    assert nxt[0] == exp and nxt[1] == nxt[2] - (nxt[2] % 256) - 768 and nxt[1] >= 225


def test_allocation_order_cap_and_exhaustion(oracle):
    """Hand-worked: bs = 2, three sequences of lengths 2, 3, 4 -> sequences 0 and 2 open a block (length a multiple of
    bs), popped from the top of the stack in batch order; with one free block left the second of them is not advanced."""
    bs = 2
    bt = np.array([[7, -1, -1, -1], [5, 6, -1, -1], [1, 2, -1, -1]], np.int32)
    sl, un = np.array([2, 3, 4], np.int32), np.array([2, 3, 4], np.int32)
    fl, fc, g = np.array([9, 8, 3, 4, -1, -1, -1, -1, -1, -1], np.int32), np.array([4], np.int32), np.array([0], np.int32)
    sel = oracle.policy_step(bt, sl, un, None, fl, fc, g, bs, 100, 4, 2)
    assert bt.tolist() == [[7, 4, -1, -1], [5, 6, -1, -1], [1, 2, 3, -1]] and int(fc[0]) == 2
    assert sl.tolist() == [3, 4, 5] and un.tolist() == [3, 4, 5] and g[0] == 1 and sel["sel_count"] == 0
    # exhaustion: one free block, two sequences need one
    bt2 = np.array([[7, -1], [5, -1]], np.int32)
    sl2, un2 = np.array([2, 2], np.int32), np.array([2, 2], np.int32)
    fl2, fc2, g2 = np.array([3, -1, -1], np.int32), np.array([1], np.int32), np.array([0], np.int32)
    sel = oracle.policy_step(bt2, sl2, un2, None, fl2, fc2, g2, bs, 100, 4, 2)
    assert sel["exhausted"] == 1 and sl2.tolist() == [3, 2] and bt2.tolist() == [[7, 3], [5, -1]] and int(fc2[0]) == 0
    # cap: five eligible sequences, max_select = 2 -> the first two in batch order
    S = 5
    bt3 = np.tile(np.arange(4, dtype=np.int32), (S, 1)) + 4 * np.arange(S, dtype=np.int32)[:, None]
    sl3, un3 = np.full(S, 7, np.int32), np.full(S, 7, np.int32)
    fl3, fc3, g3 = np.arange(20, 30, dtype=np.int32), np.array([10], np.int32), np.array([7], np.int32)
    sel = oracle.policy_step(bt3, sl3, un3, None, fl3, fc3, g3, bs, 4, 6, 2)      # g = 8 > W = 6, 8 mod 4 = 0
    assert sel["sel_count"] == 2 and sel["sel_ids"].tolist() == [0, 1] and sel["sel_win_start"].tolist() == [2, 2]
    np.testing.assert_array_equal(sel["sel_block_table"], bt3[:2])
