"""Pins of the oracle's window-query producer (kara_oracle_window_queries: PAPER.md App. C.2, reading G19) against
things other than itself: the projection against numpy's float64 matmul (a library routine), the rotary embedding against
the complex-number formulation (x_c + i x_{c+d/2}) e^{i pos f_c}, and the properties that define RoPE: identity at
position 0, norm preservation per pair, scores that depend on the relative position only."""
import numpy as np
import pytest

from conftest import bf16_bits_to_f64, f32_to_bf16_bits


def _ulp_diff(a_bits, b_bits):
    """distance in bf16 codes (sign-magnitude -> ordered integers)"""
    def key(b):
        b = b.astype(np.int32)
        return np.where(b & 0x8000, -(b & 0x7fff), b & 0x7fff)
    return np.abs(key(a_bits) - key(b_bits))


@pytest.mark.parametrize("T,Dm,Hq,d", [(5, 64, 2, 8), (17, 192, 3, 64), (9, 128, 2, 128)])
def test_projection_is_a_matmul(oracle, T, Dm, Hq, d):
    rng = np.random.default_rng(T)
    hid = f32_to_bf16_bits(rng.standard_normal((T, Dm)).astype(np.float32))
    wq = f32_to_bf16_bits((rng.standard_normal((Hq * d, Dm)) / np.sqrt(Dm)).astype(np.float32))
    got = oracle.window_queries(hid, wq, None, 10000.0, Hq, d)
    ref = bf16_bits_to_f64(hid) @ bf16_bits_to_f64(wq).T                     # library float64 matmul
    ref_bits = f32_to_bf16_bits(ref.astype(np.float32)).reshape(T, Hq, d)
    dist = _ulp_diff(got, ref_bits)
    assert dist.max() <= 1 and (dist == 0).mean() > 0.995                    # (summation order may flip a rounding tie)
    # a transposed weight or a wrong head stride would be far off
    assert np.abs(bf16_bits_to_f64(got).reshape(T, -1) - ref).max() < 2e-2 * np.abs(ref).max()


def test_rope_against_complex_formulation_and_its_properties(oracle):
    rng = np.random.default_rng(3)
    T, Dm, Hq, d, theta = 12, 64, 2, 16, 10000.0
    # an identity-like projection: hidden carries the query directly (Dm = Hq*d), wq = I
    hid_f = rng.standard_normal((T, Hq * d)).astype(np.float32)
    hid = f32_to_bf16_bits(hid_f)
    wq = f32_to_bf16_bits(np.eye(Hq * d, dtype=np.float32))
    Dm = Hq * d
    pos = np.array([0, 1, 2, 3, 7, 100, 1000, 4097, 65536, 131071, 5, 6], np.int32)
    got = bf16_bits_to_f64(oracle.window_queries(hid, wq, pos, theta, Hq, d))
    q = bf16_bits_to_f64(hid).reshape(T, Hq, d)
    f = theta ** (-2.0 * np.arange(d // 2) / d)
    z = (q[..., : d // 2] + 1j * q[..., d // 2:]) * np.exp(1j * pos[:, None, None] * f[None, None, :])
    ref = np.concatenate([z.real, z.imag], axis=-1)
    assert np.abs(got - ref).max() <= 2.0 ** -8 * np.abs(ref).max() + 1e-12   # one bf16 rounding
    # position 0: identity (exact bits)
    np.testing.assert_array_equal(got[0], q[0])
    # rotation preserves the norm of every (c, c + d/2) pair up to the output rounding
    n_in = np.hypot(q[..., : d // 2], q[..., d // 2:])
    n_out = np.hypot(got[..., : d // 2], got[..., d // 2:])
    assert np.abs(n_in - n_out).max() <= 2.0 ** -7 * n_in.max()
    # relative-position property: <RoPE(x, m), RoPE(y, n)> = <RoPE(x, m + s), RoPE(y, n + s)>
    x, y = hid[:1].copy(), hid[1:2].copy()
    def rot(v, p):
        return bf16_bits_to_f64(oracle.window_queries(v, wq, np.array([p], np.int32), theta, Hq, d))[0, 0]
    a = rot(x, 3) @ rot(y, 10)
    b = rot(x, 3 + 500) @ rot(y, 10 + 500)
    assert abs(a - b) <= 0.05 * (np.linalg.norm(q[0, 0]) * np.linalg.norm(q[1, 0]))
    # and NOT invariant when only one side moves (a dropped position would pass the line above trivially)
    assert abs(rot(x, 3) @ rot(y, 10) - rot(x, 3) @ rot(y, 40)) > 1e-3
