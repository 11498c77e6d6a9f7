"""Pins for the oracle's O4-O9 (Eq. 5-8 + App. C.3) — CPU only.

Pinned by: exact-rational budget table; hand-worked vectors (tests/golden/); the alpha=0 special
case against numpy's sort; brute force over subsets on tiny inputs (argmax-of-sum formulation,
not a re-typed sort); and the structural invariants the paper states (chunk additions <= alpha,
chunk length <= gamma incl. endpoints, |F| = keep).
"""
import itertools
import math
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest

GOLDEN = Path(__file__).parent / "golden" / "token2chunk_handworked.txt"


# ------------------------------------------------------------------------------------------
# O4 budget
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("r,n,keep", [("0.2", 56, 12), ("0.2", 480, 96), ("0.1", 992, 100),
                                      ("0.2", 992, 199), ("0.3", 992, 298), ("0.2", 1984, 397)])
def test_budget_table(oracle, r, n, keep):
    """SURVEY §8(c) O4 table; each value is ceil of an exact rational."""
    assert math.ceil(Fraction(r) * n) == keep
    assert oracle.budget(n, float(r)) == keep


def test_budget_exact_rational_sweep(oracle):
    """ceil(r n) over the paper's ranges (r in 20..60 %, W in {256,384,512,768,1024,2048},
    U in {0,32,64}) equals exact rational arithmetic — in particular
    0.2*480 must give 96, not 97 (float32 0.2f would)."""
    for pct in range(5, 101, 5):
        r = Fraction(pct, 100)
        for W in (64, 256, 384, 512, 768, 1024, 2048):
            for U in (0, 8, 32, 64):
                n = W - U
                if n <= 0:
                    continue
                assert oracle.budget(n, pct / 100) == math.ceil(r * n), (pct, n)
    assert oracle.budget(480, float(np.float32(0.2))) == 97   # the float trap the reading avoids
    assert oracle.budget(10, 1.0) == 10


# ------------------------------------------------------------------------------------------
# hand-worked vectors
# ------------------------------------------------------------------------------------------
def _parse_golden():
    cases, cur = [], None
    for line in GOLDEN.read_text().splitlines():
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tok = line.split()
        if tok[0] == "case":
            cur = {"name": tok[1]}
            cases.append(cur)
        elif tok[0] == "A":
            cur["A"] = np.array([float(x) for x in tok[1:]], np.float32)
        elif tok[0] == "I":
            cur["I"] = [int(x) for x in tok[1:]]
        elif tok[0] == "C":
            cur["C"] = [] if tok[1:] == ["-"] else [tuple(int(v) for v in x.split("-")) for x in tok[1:]]
        elif tok[0] == "F":
            cur["F"] = [int(x) for x in tok[1:]]
        else:
            cur["n"], cur["keep"], cur["alpha"], cur["gamma"] = (int(x) for x in tok)
    return cases


@pytest.mark.parametrize("case", _parse_golden(), ids=lambda c: c["name"])
def test_handworked_vectors(oracle, case):
    assert len(case["A"]) == case["n"]
    out = oracle.select(case["A"], case["keep"], case["alpha"], case["gamma"])
    assert out["I"].tolist() == case["I"]
    assert out["F"].tolist() == case["F"]
    chosen = [(int(out["I"][t]), int(out["I"][t + 1])) for t in out["chunks"] if t >= 0]
    assert chosen == case["C"]
    assert out["n_chunk_added"] == sum(b - a - 1 for a, b in case["C"])


# ------------------------------------------------------------------------------------------
# special case alpha = 0 ("w/o Token2Chunk") = plain top-keep
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,keep", [(56, 12), (480, 96), (33, 33), (7, 1)])
def test_alpha_zero_is_plain_topk(oracle, n, keep):
    rng = np.random.default_rng(n + keep)
    A = rng.random(n).astype(np.float32)
    out = oracle.select(A, keep, 0, 8)
    expect = np.sort(np.argsort(-A.astype(np.float64), kind="stable")[:keep])
    assert out["F"].tolist() == expect.tolist()
    assert out["I"].tolist() == expect.tolist()
    assert out["n_chunk_added"] == 0


def test_no_eligible_chunk_gives_plain_top_keep(oracle):
    """If no pair of consecutive candidates is closer than gamma, Token2Chunk adds nothing and
    the C.3 fill turns F into the plain top-keep set."""
    n, keep, alpha, gamma = 64, 12, 4, 3
    A = np.full(n, 0.01, np.float32) + np.arange(n, dtype=np.float32) * 1e-4
    spikes = np.arange(0, 64, 8)              # candidates 8 apart, gamma=3 => none eligible
    A[spikes] = 5.0 + np.arange(len(spikes), dtype=np.float32)
    out = oracle.select(A, keep, alpha, gamma)
    assert out["n_chunk_added"] == 0 and (out["chunks"] == -1).all()
    expect = np.sort(np.argsort(-A.astype(np.float64), kind="stable")[:keep])
    assert out["F"].tolist() == expect.tolist()


# ------------------------------------------------------------------------------------------
# brute force on tiny inputs: each TopK as an argmax over subsets
# ------------------------------------------------------------------------------------------
def _best_subset(items, size, value):
    """The size-subset of `items` with the largest total value (unique for distinct values)."""
    best, best_v = None, None
    for sub in itertools.combinations(items, size):
        v = sum(value(x) for x in sub)
        if best is None or v > best_v:
            best, best_v = sub, v
    return set(best) if best is not None else set()


def _brute_force(A, keep, alpha, gamma):
    n = len(A)
    k = keep - alpha
    P = alpha // (gamma - 2)
    Af = [Fraction(float(a)) for a in A]
    I = sorted(_best_subset(range(n), k, lambda j: Af[j]))                       # Eq. 5
    elig = [t for t in range(k - 1) if I[t + 1] - I[t] < gamma and I[t + 1] - I[t] - 1 >= 1]
    R = {t: (Af[I[t]] + Af[I[t + 1]]) * (I[t + 1] - I[t] - 1) for t in elig}     # Eq. 6
    picked = _best_subset(elig, min(P, len(elig)), lambda t: R[t])               # Eq. 7
    hat = set(I)
    for t in picked:
        hat |= set(range(I[t] + 1, I[t + 1]))                                    # Eq. 8
    rest = [j for j in range(n) if j not in hat]
    hat |= _best_subset(rest, keep - len(hat), lambda j: Af[j])                  # C.3 fill
    return I, sorted(picked), sorted(hat)


@pytest.mark.parametrize("seed", range(40))
def test_brute_force_tiny(oracle, seed):
    rng = np.random.default_rng(1000 + seed)
    n = int(rng.integers(8, 15))
    gamma = int(rng.integers(3, 6))
    keep = int(rng.integers(3, n - 1))
    alpha = int(rng.integers(0, keep))       # k = keep - alpha >= 1
    # distinct dyadic scores: sums of two and products by a small gap stay exact in fp32, and
    # subset sums are compared exactly through Fractions
    A = (rng.permutation(64)[:n].astype(np.float32) + 1) / 64
    out = oracle.select(A, keep, alpha, gamma)
    I, picked, F = _brute_force(A, keep, alpha, gamma)
    assert out["I"].tolist() == I
    # the set of chosen chunks (hence F) is unique unless two chunk subsets tie in total R;
    # a tie is decided by reading G4 (lower ordinal first), covered by the hand-worked case
    if not _has_chunk_tie(A, I, gamma, alpha):
        assert sorted(int(t) for t in out["chunks"] if t >= 0) == picked
        assert out["F"].tolist() == F


def _has_chunk_tie(A, I, gamma, alpha):
    k = len(I)
    P = alpha // (gamma - 2)
    elig = [t for t in range(k - 1) if I[t + 1] - I[t] < gamma and I[t + 1] - I[t] - 1 >= 1]
    R = [(Fraction(float(A[I[t]])) + Fraction(float(A[I[t + 1]]))) * (I[t + 1] - I[t] - 1) for t in elig]
    m = min(P, len(elig))
    tot = [sum(s) for s in itertools.combinations(R, m)] if m else []
    return len(tot) != len(set(tot)) and tot.count(max(tot)) > 1


# ------------------------------------------------------------------------------------------
# invariants at the paper's sizes
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,keep,alpha,gamma", [(56, 12, 4, 4), (480, 96, 32, 8), (480, 96, 16, 8),
                                                (992, 199, 32, 8), (1984, 397, 32, 8),
                                                (1984, 397, 112, 16), (224, 135, 32, 8)])
def test_structural_invariants(oracle, n, keep, alpha, gamma):
    rng = np.random.default_rng(n * 7 + alpha)
    A = rng.gamma(0.7, 1.0, size=n).astype(np.float32)          # skewed like real scores
    A[rng.integers(0, n, n // 10)] *= 20                         # clustered heavy hitters
    out = oracle.select(A, keep, alpha, gamma)
    I, F = out["I"], out["F"]
    k, P = keep - alpha, alpha // (gamma - 2)
    assert len(I) == k and len(F) == keep                                        # |F| = keep (G9)
    assert (np.diff(I) > 0).all() and (np.diff(F) > 0).all()                     # sorted, unique
    assert 0 <= F.min() and F.max() < n
    assert set(I.tolist()) <= set(F.tolist())                                    # I subset F
    # I is the top-k: every member outranks every non-member under (A desc, idx asc)
    out_I = np.setdiff1d(np.arange(n), I)
    assert A[I].min() >= A[out_I].max()
    chosen = [int(t) for t in out["chunks"] if t >= 0]
    assert len(chosen) <= P
    added = set()
    for t in chosen:
        a, b = int(I[t]), int(I[t + 1])
        assert b - a < gamma and b - a - 1 >= 1                                  # Eq. 7 constraint
        assert b - a + 1 <= gamma                                                # length incl. endpoints
        added |= set(range(a + 1, b))
    assert len(added) == out["n_chunk_added"] <= P * (gamma - 2) <= alpha
    assert added <= set(F.tolist())
    fill = set(F.tolist()) - set(I.tolist()) - added
    assert len(fill) == keep - k - len(added)
    unretained = np.setdiff1d(np.arange(n), F)
    if fill and len(unretained):
        assert min(A[j] for j in fill) >= A[unretained].max()                    # fill by score
    # chosen chunks outrank the eligible chunks that were not chosen
    def R(t):
        return np.float32(np.float32(A[I[t]] + A[I[t + 1]]) * np.float32(I[t + 1] - I[t] - 1))
    elig = [t for t in range(k - 1) if I[t + 1] - I[t] < gamma and I[t + 1] - I[t] - 1 >= 1]
    assert len(chosen) == min(P, len(elig))
    rest = [t for t in elig if t not in chosen]
    if chosen and rest:
        assert min(R(t) for t in chosen) >= max(R(t) for t in rest)


def test_budget_errors(oracle):
    A = np.ones(16, np.float32)
    for keep, alpha, gamma in [(4, 4, 4), (4, 5, 4), (17, 0, 4), (8, 2, 2)]:
        with pytest.raises(ValueError):
            oracle.select(A, keep, alpha, gamma)
