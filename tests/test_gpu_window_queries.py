"""The window-query producer on the GPU (kara_window_queries: PAPER.md App. C.2) against the oracle.
Tolerance: the output is a bf16 CODE decided by floating point — the oracle rounds an fp64 result once, the kernel an fp32
accumulation (d_model products, error <= d_model * 2^-24 relative to sum |terms|) followed by an fp32 rotation — so codes
may differ by ONE step where the exact value sits at a rounding boundary (near a zero crossing of the rotated value the same
absolute error spans more codes: there |got - oracle| <= 2^-15 rms is accepted).  The share of codes that flip is about
(relative error of the fp32 dot product, <~ sqrt(d_model) 2^-23) / (relative code spacing, 2^-8): at least
1 - sqrt(d_model) 2^-13 of the codes must be identical (99.8 % at d_model 256, 99.1 % at 5120).  Needs a B200."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _bits(t):
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16).copy()


def _f(bits):
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def _code(b):
    """bf16 bit patterns -> integers ordered like the values (sign-magnitude -> two's complement)"""
    b = b.astype(np.int32)
    return np.where(b & 0x8000, -(b & 0x7fff), b & 0x7fff)


def _check(got_bits, ref_bits, d_model):
    got, ref = _f(got_bits), _f(ref_bits)
    rms = np.sqrt((ref ** 2).mean())
    dist = np.abs(_code(got_bits) - _code(ref_bits))
    ok = (dist <= 1) | (np.abs(got - ref) <= 2.0 ** -15 * rms)
    assert np.all(ok), f"{int((~ok).sum())} elements more than one bf16 step from the oracle (worst {int(dist.max())} steps)"
    same = (got_bits == ref_bits).mean()
    need = 1.0 - d_model ** 0.5 * 2.0 ** -13
    assert same >= need, f"only {same:.5f} of the bf16 codes identical (need {need:.5f})"
    return same


@pytest.mark.parametrize("T,Dm,Hq,d,rope", [(200, 256, 4, 64, True), (128, 512, 2, 128, True), (333, 1024, 6, 128, True),
                                           (257, 320, 5, 64, False), (64, 64, 4, 64, True)])
def test_small_shapes_every_element(oracle, T, Dm, Hq, d, rope):
    """Ragged token counts (T not a multiple of 128), head counts that do not fill the last 256-column tile, both head sizes,
    with and without the rotary embedding; positions up to 131,071."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_01237_b200 import kara
    g = torch.Generator().manual_seed(T + Dm)
    hid = torch.randn(T, Dm, generator=g).to(torch.bfloat16)
    wq = (torch.randn(Hq * d, Dm, generator=g) / Dm ** 0.5).to(torch.bfloat16)
    pos = torch.randint(0, 131072, (T,), generator=g, dtype=torch.int32)
    pos[0], pos[1 % T] = 0, 131071
    out = kara.kara_window_queries(hid.cuda(), wq.cuda(), pos.cuda() if rope else None, 1e6, Hq, d, max_position=131071)
    torch.cuda.synchronize()
    ref = oracle.window_queries(_bits(hid), _bits(wq), pos.numpy() if rope else None, 1e6, Hq, d)
    _check(_bits(out), ref, Dm)


def test_qwen3_14b_shape_sampled_rows(oracle):
    """The producer at the bench's shape (d_model 5120, 40 heads x 128, 8,192 window tokens = 16 windows of 512): 24 sampled
    rows (first / last tile, tile edges, random) against the oracle, every head and column of those rows."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_01237_b200 import kara
    T, Dm, Hq, d = 8192, 5120, 40, 128
    dev = torch.device("cuda:0")
    g = torch.Generator(device=dev).manual_seed(7)
    hid = torch.randn(T, Dm, generator=g, device=dev).to(torch.bfloat16)
    wq = (torch.randn(Hq * d, Dm, generator=g, device=dev) / Dm ** 0.5).to(torch.bfloat16)
    pos = (torch.arange(T, device=dev, dtype=torch.int32) % 512) + 20000
    out = kara.kara_window_queries(hid, wq, pos, 1e6, Hq, d, max_position=32768)
    torch.cuda.synchronize()
    rng = np.random.default_rng(0)
    rows = sorted(set([0, 1, 127, 128, 129, 255, 4095, 4096, T - 129, T - 128, T - 1] + rng.integers(0, T, 13).tolist()))
    ref = oracle.window_queries(_bits(hid[rows]), _bits(wq), pos[rows].cpu().numpy(), 1e6, Hq, d)
    _check(_bits(out[rows]), ref, Dm)


def test_feeds_compress_window(oracle):
    """The producer's output is the window_q of kara_compress_window: project + rotate the hidden states of a small batch,
    compress with those queries on the GPU, and run the oracle's whole path on the SAME query bits: three-stage parity."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from oracle import check
    from paper_2607_01237_b200 import inputs as kin
    from paper_2607_01237_b200 import kara
    import gpu_util
    sh = kin.scaled(kin.CFG1, n_seqs=2, n_layers=1, n_q_heads=4, n_kv_heads=2, hist_lo=40, hist_hi=90)
    wl = kin.generate(sh, seed=5)
    Dm = 128
    g = torch.Generator().manual_seed(1)
    hid = torch.randn(sh.n_seqs * sh.W, Dm, generator=g).to(torch.bfloat16)
    wq = (torch.randn(sh.n_q_heads * sh.head_dim, Dm, generator=g) * (2.0 / Dm ** 0.5)).to(torch.bfloat16)
    pos = torch.cat([torch.arange(sh.W, dtype=torch.int32) + int(wl.win_start[s]) for s in range(sh.n_seqs)])
    q = kara.kara_window_queries(hid.cuda(), wq.cuda(), pos.cuda(), 1e4, sh.n_q_heads, sh.head_dim)
    torch.cuda.synchronize()
    _check(_bits(q), oracle.window_queries(_bits(hid), _bits(wq), pos.numpy(), 1e4, sh.n_q_heads, sh.head_dim), Dm)
    wl.window_q = q.view(1, sh.n_seqs, sh.W, sh.n_q_heads, sh.head_dim).cpu()
    H0 = check.host_image(wl)
    out, cache, _ = gpu_util.gpu_compress(wl)
    assert out["status"] == 0
    check.compare(H0, out, sh.n_q_heads, sh.W, sh.U, sh.ratio, sh.alpha, sh.gamma, 0, 1)
