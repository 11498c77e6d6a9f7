"""The C-ABI library builds, loads and exports every symbol include/kara.h declares — CPU only
(no compute calls: only the host-side entry points that touch no CUDA API are exercised)."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def kara():
    from paper_2607_01237_b200 import build, kara as k
    build.build()
    k.lib()
    return k


def _declared_symbols():
    text = (ROOT / "include" / "kara.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(kara_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound(kara):
    declared = _declared_symbols()
    assert len(declared) >= 14 and "kara_init_cache" in declared and "kara_compress_window" in declared \
        and "kara_gather_debug" in declared
    L = kara.lib()
    for name in declared:
        assert hasattr(L, name), f"libkara.so does not export {name}"
        assert name in kara.SYMBOLS, f"binding has no signature for {name}"
    assert sorted(kara.SYMBOLS) == declared


def test_no_torch_or_python_types_in_the_abi():
    text = (ROOT / "include" / "kara.h").read_text()
    assert 'extern "C"' in text
    code = re.sub(r"/\*.*?\*/", "", text, flags=re.S)      # declarations only, comments stripped
    assert "torch" not in code.lower() and "at::" not in code and "PyObject" not in code and "std::" not in code


def test_library_does_not_link_the_oracle(kara):
    import subprocess
    so = ROOT / "paper_2607_01237_b200" / "libkara.so"
    syms = subprocess.run(["nm", "-D", str(so)], capture_output=True, text=True).stdout
    assert "kara_oracle" not in syms


def test_budget_matches_exact_rational(kara):
    import math
    from fractions import Fraction
    for pct in range(5, 101, 5):
        for n in (56, 192, 224, 352, 480, 736, 992, 1984):
            assert kara.kara_budget(n, pct / 100) == math.ceil(Fraction(pct, 100) * n)
    assert kara.kara_budget(0, 0.2) < 0 and kara.kara_budget(10, 0.0) < 0 and kara.kara_budget(10, 1.5) < 0


def test_init_cache_geometry_and_errors(kara):
    L = kara.lib()
    h = L.kara_init_cache(16, 40, 8, 128)
    assert h
    assert L.kara_block_bytes(h) == 40 * 8 * 16 * 128 * 2
    assert L.kara_pool_bytes(h, 1000) == 40 * 1000 * 8 * 16 * 128 * 2
    ws = L.kara_workspace_bytes(h, 40, 1, 40, 512, 32, 0.2, 32)
    assert ws > 320 * 480 * 4 and ws % 256 == 0
    assert L.kara_last_launch_count(h) == 0 and L.kara_last_score_path(h) == 0
    # compress before attach is an argument error, not a crash
    rc = L.kara_compress_window(h, 0, 1, 1, 1, 1, 1, None, 1, 40, 512, 32, 0.2, 32, 8, 0, 1, 0, None)
    assert rc == kara.KARA_EINVAL and b"attach" in L.kara_last_error()
    rc = L.kara_compress_window(h, 0, 1, 1, 1, 1, 1, None, 1, 40, 512, 32, 0.2, 96, 8, 0, 1, 0, None)
    assert rc == kara.KARA_EBUDGET
    L.kara_destroy(h)
    for bad in [(15, 1, 1, 128), (16, 1, 1, 96), (512, 1, 1, 128), (16, 0, 1, 128)]:
        assert not L.kara_init_cache(*bad)
        assert L.kara_last_error() != b""


def test_binding_fails_loudly_without_the_library(kara, monkeypatch, tmp_path):
    monkeypatch.setattr(kara, "_LIB", None)
    monkeypatch.setattr(kara, "_SO", tmp_path / "missing.so")
    with pytest.raises(kara.KaraError):
        kara.lib()


def test_header_constants_match_the_binding(kara):
    """Every #define of include/kara.h (flags, debug selectors, status bits, error codes) has the same value in the
    Python binding: the binding marshals arguments, it must not reinterpret them."""
    text = (ROOT / "include" / "kara.h").read_text()
    defs = dict(re.findall(r"^#define\s+(KARA_[A-Z0-9_]+)\s+\(?(-?\d+)u?\)?", text, flags=re.M))
    assert {"KARA_COMMIT", "KARA_KEEP_DEBUG", "KARA_SCORE_QBUF_ONLY", "KARA_SCORE_SIMT"} <= set(defs)
    checked = 0
    for name, val in defs.items():
        if hasattr(kara, name):
            assert getattr(kara, name) == int(val), name
            checked += 1
    assert checked >= 10


def test_new_entry_points_check_their_arguments_on_the_host(kara):
    """kara_compress_windows, kara_policy_step / _commit and kara_window_queries validate their arguments before any CUDA
    call: errors are codes + messages, never crashes (no GPU needed)."""
    L = kara.lib()
    h = L.kara_init_cache(16, 2, 2, 64)
    assert L.kara_compress_windows(h, 0, 1, 1, 1, 1, 1, None, 0, 1, 4, 64, 8, 0.2, 4, 4, 0, 1, 0, None) == kara.KARA_EINVAL
    assert b"n_windows" in L.kara_last_error()
    # policy calls need an attached pool / non-null state
    assert L.kara_policy_step(h, 4, 1, 8, 1, 1, None, 1, 8, 64, 2, 1, 1, 1, 1, 1, 1, None) == kara.KARA_EINVAL
    assert b"attach" in L.kara_last_error() or b"pool" in L.kara_last_error()
    assert L.kara_policy_commit(h, 2, None, None, None, None, None, 64, 8, 0.2, None, 8, None, None, None) == kara.KARA_EINVAL
    assert L.kara_policy_commit(h, 2, 1, 1, 1, 1, 1, 64, 80, 0.2, 1, 8, 1, 1, None) == kara.KARA_EINVAL     # W <= U
    L.kara_destroy(h)
    # the producer: shapes it does not take, alignment, missing workspace for the rotary tables
    assert L.kara_window_queries(None, None, None, 0, 1e4, 4, 64, 2, 64, None, None, 0, None) == kara.KARA_EINVAL
    assert L.kara_window_queries(16, 16, None, 0, 1e4, 4, 64, 2, 96, 16, None, 0, None) == kara.KARA_EUNSUPPORTED
    assert L.kara_window_queries(16, 16, None, 0, 1e4, 4, 100, 2, 64, 16, None, 0, None) == kara.KARA_EUNSUPPORTED
    assert L.kara_window_queries(16, 24, None, 0, 1e4, 4, 64, 2, 64, 16, None, 0, None) == kara.KARA_EINVAL      # alignment
    assert L.kara_window_queries(16, 16, 16, 100, 1e4, 4, 64, 2, 64, 16, None, 0, None) == kara.KARA_EINVAL      # no workspace
    assert L.kara_window_queries_workspace_bytes(131071, 128) == 8 * ((131071 >> 8) + 1 + 256) * 64
    assert L.kara_window_queries_workspace_bytes(100, 96) == 0


def test_static_scratch_entry_point_refuses_oversized_tables_on_the_host(kara):
    """kara_window_queries_static (no device allocation: rotary tables in the library's built-in array) rejects a
    max_position whose tables exceed KARA_STATIC_SCRATCH_BYTES before any CUDA call, with the limit in the message."""
    L = kara.lib()
    for d, limit in ((128, 458751), (64, 983039)):
        assert L.kara_window_queries_workspace_bytes(limit, d) == kara.KARA_STATIC_SCRATCH_BYTES
        rc = L.kara_window_queries_static(16, 16, 16, limit + 1, 1e4, 4, 64, 2, d, 16, None)
        assert rc == kara.KARA_ENOMEM
        msg = L.kara_last_error().decode()
        assert str(kara.KARA_STATIC_SCRATCH_BYTES) in msg and str(limit) in msg and "kara_window_queries" in msg
    # without positions no scratch is involved: the call is the workspace variant's, argument checks included
    assert L.kara_window_queries_static(None, None, None, 0, 1e4, 4, 64, 2, 64, None, None) == kara.KARA_EINVAL
    assert L.kara_window_queries_static(16, 16, None, 0, 1e4, 4, 64, 2, 96, 16, None) == kara.KARA_EUNSUPPORTED


def test_workspace_reserves_strips_for_the_packed_buffer_tiles(kara):
    """KARA_SCORE_QBUF_ONLY can cut a unit into more query tiles than the full window has (W = 100, U = 65, G = 3: 4 against
    3), and with few units every tile is a cluster of its own: kara_workspace_bytes must reserve 4 partial-score strips per
    unit.  2 units, n = 35 (padded to 36), k = 3, keep = 7: status 256 + partial 4 B x 2 x 4 x 36 = 1152 -> 1280 +
    scores 288 -> 512 + I 256 + F 256 bytes."""
    L = kara.lib()
    h = L.kara_init_cache(16, 1, 2, 64)
    assert L.kara_workspace_bytes(h, 1, 1, 6, 100, 65, 0.2, 4) == 256 + 1280 + 512 + 256 + 256
    # where the packed variant has fewer tiles nothing changes: 2 units x 1 strip bound by the full window's 3 tiles
    assert L.kara_workspace_bytes(h, 1, 1, 6, 100, 5, 0.2, 4) == 256 + 4 * 2 * 3 * 96 + 768 + 256 + 256
    L.kara_destroy(h)
