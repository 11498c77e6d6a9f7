"""kara_window_queries_static — the window-query producer for callers that may not allocate device memory (a serving
engine in the middle of decoding has put all of its HBM into the KV pool: a cudaMalloc there fails or stalls the device, and
its allocator policy forbids one) — against kara_window_queries with a caller-owned workspace, on the same inputs.

The two entry points run the same table kernel and the same GEMM and differ only in where the rotary tables live (the
library's built-in 1 MiB device array instead of a workspace), so their outputs should be the same bits; what is asserted is
the tolerance of tests/test_gpu_window_queries.py (every bf16 code within ONE step or 2^-15 rms, at least
1 - sqrt(d_model) 2^-13 of them identical).  Two calls in a row with different theta / head_dim / max_position: the array
keeps the first call's tables, and the second call must not see them.

This file is named to be collected last (pytest -x would hide every later test behind a failure here); it passes alone in a
fresh process (its first call then does the per-device address lookup) and after the other tests.  Needs a B200."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _bits(t):
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16).copy()


def _values(bits):
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def _order(bits):
    """bf16 bit patterns -> integers ordered like the values they encode"""
    b = bits.astype(np.int32)
    return np.where(b & 0x8000, -(b & 0x7fff), b & 0x7fff)


def _assert_same_within_tolerance(got_bits, want_bits, d_model, what):
    got, want = _values(got_bits), _values(want_bits)
    rms = np.sqrt((want ** 2).mean())
    steps = np.abs(_order(got_bits) - _order(want_bits))
    ok = (steps <= 1) | (np.abs(got - want) <= 2.0 ** -15 * rms)
    assert np.all(ok), f"{what}: {int((~ok).sum())} elements more than one bf16 step apart (worst {int(steps.max())} steps)"
    same = (got_bits == want_bits).mean()
    need = 1.0 - d_model ** 0.5 * 2.0 ** -13
    assert same >= need, f"{what}: only {same:.5f} of the bf16 codes identical (need {need:.5f})"


# (T, d_model, n_q_heads, head_dim, theta, max_position): the second call uses smaller tables with another layout
CALLS = [(333, 1024, 6, 128, 1e6, 131071), (200, 256, 4, 64, 1e4, 40959)]


def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_01237_b200 import kara
    dev = torch.device("cuda:0")
    cases = []
    for T, Dm, Hq, d, theta, max_pos in CALLS:
        g = torch.Generator().manual_seed(T + Dm)
        hid = torch.randn(T, Dm, generator=g).to(torch.bfloat16).to(dev)
        wq = (torch.randn(Hq * d, Dm, generator=g) / Dm ** 0.5).to(torch.bfloat16).to(dev)
        pos = torch.randint(0, max_pos + 1, (T,), generator=g, dtype=torch.int32)
        pos[0], pos[1] = 0, max_pos
        pos = pos.to(dev)
        # the existing path (workspace allocated by the binding) first: its result is what the new entry point must give
        want = kara.kara_window_queries(hid, wq, pos, theta, Hq, d, max_position=max_pos)
        out = torch.full((T, Hq, d), float("nan"), dtype=torch.bfloat16, device=dev)     # every element must be written
        cases.append((hid, wq, pos, theta, Hq, d, max_pos, Dm, want, out))
    torch.cuda.synchronize()

    # two calls in a row on one stream, nothing in between
    for i, (hid, wq, pos, theta, Hq, d, max_pos, Dm, want, out) in enumerate(cases):
        if i == 1:
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info(dev)[0]
        kara.kara_window_queries_static(hid, wq, pos, theta, Hq, d, out, max_pos)
    torch.cuda.synchronize()
    # once the first call has loaded the kernels, a call takes no device memory
    assert torch.cuda.mem_get_info(dev)[0] >= free_before

    for i, (hid, wq, pos, theta, Hq, d, max_pos, Dm, want, out) in enumerate(cases):
        _assert_same_within_tolerance(_bits(out), _bits(want), Dm, f"call {i + 1}")

    # ... and once more in the other order, over the tables the calls above left behind
    for hid, wq, pos, theta, Hq, d, max_pos, Dm, want, out in reversed(cases):
        out.fill_(float("nan"))
        kara.kara_window_queries_static(hid, wq, pos, theta, Hq, d, out, max_pos)
    torch.cuda.synchronize()
    for i, (hid, wq, pos, theta, Hq, d, max_pos, Dm, want, out) in enumerate(cases):
        _assert_same_within_tolerance(_bits(out), _bits(want), Dm, f"call {i + 1}, second round")


def test_static_scratch_without_positions_and_beyond_the_limit():
    """No rotary embedding: no scratch is touched and the result is the workspace path's.  A max_position whose tables do not
    fit the built-in array is refused with KARA_ENOMEM and a message that names the limit; the output is left alone."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_01237_b200 import kara
    dev = torch.device("cuda:0")
    T, Dm, Hq, d = 257, 320, 5, 64
    g = torch.Generator().manual_seed(3)
    hid = torch.randn(T, Dm, generator=g).to(torch.bfloat16).to(dev)
    wq = (torch.randn(Hq * d, Dm, generator=g) / Dm ** 0.5).to(torch.bfloat16).to(dev)
    want = kara.kara_window_queries(hid, wq, None, 1e4, Hq, d)
    out = torch.full((T, Hq, d), float("nan"), dtype=torch.bfloat16, device=dev)
    kara.kara_window_queries_static(hid, wq, None, 1e4, Hq, d, out, 0)
    torch.cuda.synchronize()
    _assert_same_within_tolerance(_bits(out), _bits(want), Dm, "no rotary embedding")

    pos = torch.zeros(T, dtype=torch.int32, device=dev)
    out.zero_()
    limit = (kara.KARA_STATIC_SCRATCH_BYTES // (4 * d) - 256) * 256 - 1
    kara.kara_window_queries_static(hid, wq, pos, 1e4, Hq, d, out, limit)          # the largest max_position that fits
    with pytest.raises(kara.KaraError) as err:
        kara.kara_window_queries_static(hid, wq, pos, 1e4, Hq, d, out.zero_(), limit + 1)
    assert err.value.code == kara.KARA_ENOMEM and str(kara.KARA_STATIC_SCRATCH_BYTES) in str(err.value)
    torch.cuda.synchronize()
    assert not out.any(), "a refused call must not write its output"
