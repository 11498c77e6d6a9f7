"""The periodic compression policy on the device (kara_policy_step / kara_policy_commit, Alg. 1 + App. C.4) against
the oracle, as a whole decoding loop: every step both sides advance the running queue (allocation from the free list
included); at every compression event the selected sub-batch goes through kara_compress_window on the GPU and through the
oracle's O1-O11 on the host image, with the three-stage parity check of oracle/check.py; then both commit.  All integer
state — block tables, lengths, counters, the free list and its order, the selection — is compared bit for bit after EVERY
step, every pool byte after every event.  Needs a B200."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("bs,W,U,delta,m,S,steps,seed", [(16, 64, 8, 8, 3, 6, 260, 1), (32, 128, 16, 16, 2, 5, 420, 2),
                                                         (16, 48, 0, 5, 4, 300, 140, 3)])
def test_decoding_loop_with_policy_and_compression(oracle, bs, W, U, delta, m, S, steps, seed):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from oracle import check
    from paper_2607_01237_b200 import kara
    import gpu_util
    kara.lib()
    dev = torch.device("cuda:0")
    L, Hq, Hkv, d, ratio, alpha, gamma = 2, 4, 2, 64, 0.25, 4, 4
    n = W - U
    keep = oracle.budget(n, ratio)
    max_blocks = (steps + bs - 1) // bs + 2
    NB = S * 5 if S > 50 else S * max_blocks             # the big batch runs into pool exhaustion on purpose
    g = torch.Generator().manual_seed(seed)
    k_pool = torch.randn(L, NB, Hkv, bs, d, generator=g).to(torch.bfloat16)
    v_pool = torch.randn(L, NB, Hkv, bs, d, generator=g).to(torch.bfloat16)
    rng = np.random.default_rng(seed)
    # host state (oracle side)
    H = dict(k=check.bits(k_pool), v=check.bits(v_pool), bt=np.full((S, max_blocks), -1, np.int32),
             sl=np.zeros(S, np.int32), un=np.zeros(S, np.int32), fl=rng.permutation(NB).astype(np.int32),
             fc=np.array([NB], np.int32), g=np.zeros(1, np.int32))
    # device state
    D = dict(k=k_pool.to(dev), v=v_pool.to(dev), bt=torch.from_numpy(H["bt"]).to(dev), sl=torch.from_numpy(H["sl"]).to(dev),
             un=torch.from_numpy(H["un"]).to(dev), fl=torch.from_numpy(H["fl"]).to(dev), fc=torch.from_numpy(H["fc"]).to(dev),
             g=torch.zeros(1, dtype=torch.int32, device=dev), exh=torch.zeros(1, dtype=torch.int32, device=dev))
    sel = dict(ids=torch.empty(m, dtype=torch.int32, device=dev), count=torch.zeros(1, dtype=torch.int32, device=dev),
               block_table=torch.empty(m, max_blocks, dtype=torch.int32, device=dev),
               seq_lens=torch.empty(m, dtype=torch.int32, device=dev), win_start=torch.empty(m, dtype=torch.int32, device=dev))
    cache = kara.KaraCache(bs, L, Hkv, d)
    cache.attach_pool(D["k"], D["v"], D["fl"], D["fc"])
    events = exhausted = 0
    for step in range(steps):
        active = (rng.random(S) < 0.92).astype(np.uint8)
        # ---- one decoding step of Alg. 1 on both sides ----
        o = oracle.policy_step(H["bt"], H["sl"], H["un"], active, H["fl"], H["fc"], H["g"], bs, delta, W, m)
        exhausted += o["exhausted"]
        cache.policy_step(D["bt"], D["sl"], D["un"], torch.from_numpy(active).to(dev), D["g"], delta, W, sel, D["exh"])
        torch.cuda.synchronize()
        cnt = int(sel["count"][0])
        assert cnt == o["sel_count"]
        np.testing.assert_array_equal(sel["ids"].cpu().numpy(), o["sel_ids"])
        np.testing.assert_array_equal(sel["seq_lens"].cpu().numpy(), o["sel_seq_lens"])
        np.testing.assert_array_equal(sel["win_start"].cpu().numpy(), o["sel_win_start"])
        np.testing.assert_array_equal(sel["block_table"].cpu().numpy(), o["sel_block_table"])
        if cnt:
            events += 1
            # ---- the compression event on the selected sub-batch (rows >= cnt are absent: skipped silently) ----
            q = torch.randn(L, m, W, Hq, d, generator=g).to(torch.bfloat16)
            H0 = dict(k=H["k"], v=H["v"], q=check.bits(q[:, :cnt]), bt=o["sel_block_table"][:cnt].copy(),
                      sl=o["sel_seq_lens"][:cnt].copy(), ws=o["sel_win_start"][:cnt].copy(), fl=H["fl"], fc=H["fc"])
            cache.compress_window(0, L, sel["block_table"], sel["seq_lens"], sel["win_start"], q.to(dev), W, U, ratio, alpha,
                                  gamma, kara.KARA_COMMIT | kara.KARA_KEEP_DEBUG)
            torch.cuda.synchronize()
            Dv = dict(k=D["k"], v=D["v"], bt=sel["block_table"][:cnt], sl=sel["seq_lens"][:cnt], fl=D["fl"], fc=D["fc"])
            out = gpu_util.readback(cache, Dv, 0, L, cnt, Hkv, kara.KARA_KEEP_DEBUG)
            assert out["status"] == 0 and cache.last_score_path() == 2
            check.compare(H0, out, Hq, W, U, ratio, alpha, gamma, 0, L, commit=True)          # S1, S2, S3
            # the oracle's state moves on FROM THE GPU'S SCORES (stage S2), so both sides stay bit-identical
            Hs = {k_: v_ for k_, v_ in H0.items()}
            check.run_oracle(Hs, Hq, W, U, ratio, alpha, gamma, 0, L, True, scores_in=np.ascontiguousarray(out["scores"]))
            o["sel_block_table"][:cnt], o["sel_seq_lens"][:cnt] = Hs["bt"], Hs["sl"]
            oracle.policy_commit(o, keep, U, H["bt"], H["sl"], H["un"])
            cache.policy_commit(sel, W, U, ratio, D["bt"], D["sl"], D["un"])
            torch.cuda.synchronize()
            np.testing.assert_array_equal(check.bits(D["k"]), H["k"])
            np.testing.assert_array_equal(check.bits(D["v"]), H["v"])
        # ---- all integer state after every step ----
        np.testing.assert_array_equal(D["bt"].cpu().numpy(), H["bt"])
        np.testing.assert_array_equal(D["sl"].cpu().numpy(), H["sl"])
        np.testing.assert_array_equal(D["un"].cpu().numpy(), H["un"])
        assert int(D["fc"][0]) == int(H["fc"][0]) and int(D["g"][0]) == int(H["g"][0]) == step + 1
        np.testing.assert_array_equal(D["fl"].cpu().numpy()[: int(H["fc"][0])], H["fl"][: int(H["fc"][0])])
        assert int(D["exh"][0]) == exhausted
    assert events >= 3
    if S > 50:
        assert exhausted > 0                  # the small pool ran dry: those sequences were not advanced, on both sides
    live = np.concatenate([H["bt"][s][H["bt"][s] >= 0] for s in range(S)])
    assert sorted(np.concatenate([live, H["fl"][: int(H["fc"][0])]]).tolist()) == list(range(NB))


def test_policy_commit_leaves_a_skipped_sequence_alone():
    """kara_policy_commit (include/kara.h): a sub-batch row that kara_compress_window skipped because of a fault comes back
    with the length it went in with; committing it would set `uncompressed` to U + t as if its window had been compressed.
    Two selected rows, the first compressed (shorter by W - keep - U), the second returned unchanged: the first sequence
    takes the sub-batch's table row, length and U + t, the second keeps its table row, length and counter."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_01237_b200 import kara
    dev = torch.device("cuda:0")
    W, U, ratio, max_blocks = 64, 8, 0.25, 12
    keep = kara.kara_budget(W - U, ratio)                         # 14
    i32 = dict(dtype=torch.int32, device=dev)
    bt = torch.arange(4 * max_blocks, **i32).reshape(4, max_blocks).contiguous()
    sl = torch.tensor([150, 90, 170, 40], **i32)
    un = torch.tensor([70, 66, 75, 40], **i32)
    # sequences 2 and 1 were selected, in that order; window starts 100 and 20, tails t = 170-100-64 = 6 and 90-20-64 = 6
    sel = dict(ids=torch.tensor([2, 1, -1], **i32), count=torch.tensor([2], **i32),
               block_table=torch.full((3, max_blocks), -7, **i32), win_start=torch.tensor([100, 20, 0], **i32),
               seq_lens=torch.tensor([170 - (W - keep - U), 90, -1], **i32))
    bt0, sl0, un0 = bt.clone(), sl.clone(), un.clone()
    h = kara.KaraCache(16, 1, 1, 64)
    h.policy_commit(sel, W, U, ratio, bt, sl, un)
    torch.cuda.synchronize()
    assert sl.tolist() == [150, 90, 170 - (W - keep - U), 40]
    assert un.tolist() == [70, 66, U + 6, 40]
    assert (bt[2] == -7).all()
    for s in (0, 1, 3):
        assert torch.equal(bt[s], bt0[s])
