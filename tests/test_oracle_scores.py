"""Pins for the oracle's O1-O3 (Eq. 4) — CPU only.

The oracle is plain C loops; here it is pinned to things other than itself:
  * a library route: float64 matmul + scipy.special.softmax + sum (special case: Eq. 4 IS
    colsum(softmax(QK^T/sqrt d)));
  * closed forms (Q=0, equal keys, one-hot), invariants (sum_j A_j = G*W) and equivariances,
    chosen so that a dropped 1/sqrt(d), a softmax over the wrong axis, a transposed operand, a
    missing GQA head or a buffer-key leak fails at least one of them.
"""
import numpy as np
import pytest
from scipy.special import softmax

from conftest import bf16_bits_to_f64, f32_to_bf16_bits


def _rand_unit(rng, W, G, n, d, qscale=1.0, kscale=1.0):
    q = f32_to_bf16_bits(rng.standard_normal((W, G, d)).astype(np.float32) * qscale)
    k = f32_to_bf16_bits(rng.standard_normal((n, d)).astype(np.float32) * kscale)
    return q, k


def _library_scores(q_bits, k_bits):
    """float64 library restatement of Eq. 4 on the widened bf16 values."""
    W, G, d = q_bits.shape
    q = bf16_bits_to_f64(q_bits).reshape(W * G, d)
    k = bf16_bits_to_f64(k_bits)
    p = softmax(q @ k.T / np.sqrt(d), axis=1)      # softmax over the key dimension
    return p.sum(axis=0)                           # colsum over all queries


@pytest.mark.parametrize("W,G,n,d", [(64, 4, 56, 64), (32, 5, 24, 128), (17, 1, 17, 32),
                                     (40, 8, 33, 128), (8, 2, 1, 16)])
def test_matches_library_softmax(oracle, W, G, n, d):
    rng = np.random.default_rng(W * 1000 + n)
    q, k = _rand_unit(rng, W, G, n, d, qscale=1.5, kscale=2.0)
    A64, A32 = oracle.scores(q, k)
    ref = _library_scores(q, k)
    np.testing.assert_allclose(A64, ref, rtol=1e-12, atol=0)
    np.testing.assert_allclose(A32, ref, rtol=1.2e-7)   # rounded once to fp32


def test_bf16_widening_is_exact(oracle):
    bits = np.array([0x0000, 0x8000, 0x3F80, 0xBF80, 0x4049, 0x0001, 0x7F7F, 0x3DCD], np.uint16)
    got = np.array([oracle.lib().kara_oracle_bf16_to_double(int(b)) for b in bits])
    np.testing.assert_array_equal(got, bf16_bits_to_f64(bits))
    assert got[2] == 1.0 and got[3] == -1.0 and got[4] == 3.140625


@pytest.mark.parametrize("W,G,n,d", [(64, 4, 56, 64), (16, 5, 48, 128)])
def test_rows_sum_to_one_invariant(oracle, W, G, n, d):
    """Each softmax row sums to 1 => sum_j A_j = G*W, and 0 < A_j <= G*W."""
    rng = np.random.default_rng(7)
    q, k = _rand_unit(rng, W, G, n, d, qscale=3.0, kscale=3.0)
    A64, A32 = oracle.scores(q, k)
    assert abs(A64.sum() - G * W) < 1e-9 * G * W
    assert (A64 > 0).all() and (A64 <= G * W).all()
    np.testing.assert_allclose(A32, A64, rtol=6e-8)


def test_zero_queries_give_uniform_scores(oracle):
    """Q = 0 => every logit is 0 => p = 1/n => A_j = G*W/n exactly representable here."""
    W, G, n, d = 32, 4, 16, 64
    rng = np.random.default_rng(3)
    _, k = _rand_unit(rng, W, G, n, d)
    q = np.zeros((W, G, d), np.uint16)
    A64, _ = oracle.scores(q, k)
    np.testing.assert_array_equal(A64, np.full(n, G * W / n))


def test_equal_keys_give_uniform_scores(oracle):
    W, G, n, d = 24, 2, 12, 32
    rng = np.random.default_rng(4)
    q, k = _rand_unit(rng, W, G, n, d)
    k[:] = k[0]
    A64, _ = oracle.scores(q, k)
    np.testing.assert_allclose(A64, np.full(n, G * W / n), rtol=1e-14)


def test_one_hot_construction_counts_queries(oracle):
    """K_j = c*e_j, Q_i = c*e_{pi(i)} with c large: logit = c^2/sqrt(d) on the matching key, 0
    elsewhere => p -> one-hot => A_j -> #{(i,g): pi(i,g) = j}."""
    W, G, n, d = 20, 3, 8, 16
    rng = np.random.default_rng(5)
    c = 32.0
    k = np.zeros((n, d), np.float32)
    k[np.arange(n), np.arange(n)] = c
    pi = rng.integers(0, n, size=(W, G))
    q = np.zeros((W, G, d), np.float32)
    for i in range(W):
        for g in range(G):
            q[i, g, pi[i, g]] = c
    A64, _ = oracle.scores(f32_to_bf16_bits(q), f32_to_bf16_bits(k))
    counts = np.bincount(pi.ravel(), minlength=n).astype(np.float64)
    # off-target mass per row is (n-1)*exp(-c^2/sqrt(d)) = 7*exp(-256) ~ 0
    np.testing.assert_allclose(A64, counts, atol=1e-100)


def test_scale_is_one_over_sqrt_d(oracle):
    """Two keys, one query: A = softmax([q.k0, q.k1]/sqrt(d)) in closed form — catches a
    missing or wrong temperature."""
    d = 64
    q = np.zeros((1, 1, d), np.float32); q[0, 0, 0] = 4.0
    k = np.zeros((2, d), np.float32); k[0, 0] = 2.0; k[1, 0] = -1.0
    A64, _ = oracle.scores(f32_to_bf16_bits(q), f32_to_bf16_bits(k))
    s = np.array([8.0, -4.0]) / 8.0
    expect = np.exp(s) / np.exp(s).sum()
    np.testing.assert_allclose(A64, expect, rtol=1e-15)


def test_key_permutation_equivariance_and_query_invariance(oracle):
    W, G, n, d = 16, 4, 24, 64
    rng = np.random.default_rng(6)
    q, k = _rand_unit(rng, W, G, n, d, qscale=2.0)
    A64, _ = oracle.scores(q, k)
    perm = rng.permutation(n)
    A_perm, _ = oracle.scores(q, np.ascontiguousarray(k[perm]))
    np.testing.assert_allclose(A_perm, A64[perm], rtol=1e-13)
    # permuting query rows (tokens, and heads inside the group) leaves A unchanged
    qp = np.ascontiguousarray(q[rng.permutation(W)][:, rng.permutation(G)])
    A_q, _ = oracle.scores(qp, k)
    np.testing.assert_allclose(A_q, A64, rtol=1e-13)


def test_common_key_shift_invariance(oracle):
    """Adding one vector v to every key adds q.v to a whole row of logits; softmax rows are
    shift-invariant.  Uses small integers so bf16 holds K+v exactly."""
    W, G, n, d = 12, 2, 10, 32
    rng = np.random.default_rng(8)
    q = rng.integers(-3, 4, size=(W, G, d)).astype(np.float32) / 4
    k = rng.integers(-4, 5, size=(n, d)).astype(np.float32) / 2
    v = rng.integers(-4, 5, size=(d,)).astype(np.float32) / 2
    A0, _ = oracle.scores(f32_to_bf16_bits(q), f32_to_bf16_bits(k))
    A1, _ = oracle.scores(f32_to_bf16_bits(q), f32_to_bf16_bits(k + v))
    np.testing.assert_allclose(A1, A0, rtol=1e-12)


def test_gqa_group_is_summed_not_averaged(oracle):
    """Reading G1: the G query heads sharing a KV head are summed with the window queries."""
    W, G, n, d = 8, 4, 6, 32
    rng = np.random.default_rng(9)
    q, k = _rand_unit(rng, W, G, n, d)
    A_all, _ = oracle.scores(q, k)
    parts = [oracle.scores(np.ascontiguousarray(q[:, g:g + 1]), k)[0] for g in range(G)]
    np.testing.assert_allclose(A_all, np.sum(parts, axis=0), rtol=1e-13)


def test_strided_query_access(oracle):
    """The C entry point reads (i,g) at q + i*tok_stride + g*head_stride: score one KV-head
    group out of a [W, Hq, d] tensor without copying and compare with the sliced copy."""
    import ctypes as C
    W, Hq, Hkv, n, d = 10, 6, 2, 7, 16
    G = Hq // Hkv
    rng = np.random.default_rng(10)
    qfull = f32_to_bf16_bits(rng.standard_normal((W, Hq, d)).astype(np.float32))
    k = f32_to_bf16_bits(rng.standard_normal((n, d)).astype(np.float32))
    for hk in range(Hkv):
        ref, _ = oracle.scores(np.ascontiguousarray(qfull[:, hk * G:(hk + 1) * G]), k)
        A = np.empty(n, np.float64)
        base = qfull.ctypes.data + 2 * hk * G * d
        rc = oracle.lib().kara_oracle_scores(
            C.cast(base, C.POINTER(C.c_uint16)), Hq * d, d,
            k.ctypes.data_as(C.POINTER(C.c_uint16)), d, W, G, n, d,
            A.ctypes.data_as(C.POINTER(C.c_double)), None)
        assert rc == 0
        np.testing.assert_array_equal(A, ref)


def test_buffer_only_ablation_uses_last_U_queries(oracle):
    """'w/o Bi-Attention': queries from the buffer U only."""
    W, U, G, n, d = 24, 8, 2, 16, 32
    rng = np.random.default_rng(11)
    q, k = _rand_unit(rng, W, G, n, d)
    A_buf, _ = oracle.scores(q, k, buffer_only_U=U)
    ref = _library_scores(np.ascontiguousarray(q[W - U:]), k)
    np.testing.assert_allclose(A_buf, ref, rtol=1e-12)
    assert abs(A_buf.sum() - G * U) < 1e-9


def test_heavy_tailed_logits_are_stable(oracle):
    """Student-t-like keys: |logit| ~ 80, within-row range ~ 90 (SURVEY §7 hard part 10).  The
    max-subtracted softmax must neither overflow nor lose the row normalisation."""
    W, G, n, d = 8, 2, 32, 128
    rng = np.random.default_rng(12)
    q = rng.standard_normal((W, G, d)).astype(np.float32) * 3
    k = (rng.standard_t(3, size=(n, d)) * 6).astype(np.float32)
    qb, kb = f32_to_bf16_bits(q), f32_to_bf16_bits(k)
    A64, _ = oracle.scores(qb, kb)
    assert np.isfinite(A64).all()
    np.testing.assert_allclose(A64, _library_scores(qb, kb), rtol=1e-11, atol=1e-300)
    assert abs(A64.sum() - G * W) < 1e-9 * G * W
