"""ctypes access to the CPU oracle (oracle/kara_oracle.c).

TEST INFRASTRUCTURE ONLY — see the header of kara_oracle.h.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It imports nothing from the product package and the product imports nothing from here.

`build()` compiles the C file with gcc (-O2, no fast-math, no FP contraction) into
oracle/libkara_oracle.so; `lib()` loads it (building on demand).  The wrappers below only
marshal numpy arrays; every step of the method runs in the C code.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "kara_oracle.c"
_HDR = _HERE / "kara_oracle.h"
_SO = _HERE / "libkara_oracle.so"
_LIB = None

OK, EINVAL, EBUDGET = 0, -1, -2


def build(force: bool = False) -> Path:
    """gcc -O2 -std=c99 -ffp-contract=off -shared -fPIC kara_oracle.c -o libkara_oracle.so"""
    newest = max(_SRC.stat().st_mtime, _HDR.stat().st_mtime)
    if force or not _SO.exists() or _SO.stat().st_mtime < newest:
        tmp = _SO.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-Wextra",
               "-shared", "-fPIC", str(_SRC), "-o", str(tmp), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _SO)
    return _SO


class Layout(C.Structure):
    _fields_ = [("block_size", C.c_int), ("n_layers", C.c_int), ("n_kv_heads", C.c_int),
                ("head_dim", C.c_int), ("sL", C.c_long), ("sB", C.c_long), ("sH", C.c_long),
                ("sS", C.c_long), ("num_blocks", C.c_long)]


def lib() -> C.CDLL:
    global _LIB
    if _LIB is None:
        L = C.CDLL(str(build()))
        u16p, f32p, f64p, i32p = (C.POINTER(C.c_uint16), C.POINTER(C.c_float),
                                  C.POINTER(C.c_double), C.POINTER(C.c_int32))
        L.kara_oracle_bf16_to_double.restype = C.c_double
        L.kara_oracle_bf16_to_double.argtypes = [C.c_uint16]
        L.kara_oracle_budget.restype = C.c_int
        L.kara_oracle_budget.argtypes = [C.c_int, C.c_double]
        L.kara_oracle_scores.restype = C.c_int
        L.kara_oracle_scores.argtypes = [u16p, C.c_long, C.c_long, u16p, C.c_long,
                                         C.c_int, C.c_int, C.c_int, C.c_int, f64p, f32p]
        L.kara_oracle_scores_buffer_queries.restype = C.c_int
        L.kara_oracle_scores_buffer_queries.argtypes = [u16p, C.c_long, C.c_long, u16p, C.c_long,
                                                        C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                                        f64p, f32p]
        L.kara_oracle_select.restype = C.c_int
        L.kara_oracle_select.argtypes = [f32p, C.c_int, C.c_int, C.c_int, C.c_int,
                                         i32p, i32p, i32p, i32p]
        L.kara_oracle_compact_rows.restype = C.c_int
        L.kara_oracle_compact_rows.argtypes = [u16p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                               i32p, C.c_int, u16p]
        L.kara_oracle_metadata.restype = C.c_int
        L.kara_oracle_metadata.argtypes = [C.c_int, C.c_int, C.c_int, i32p, i32p, i32p,
                                           C.c_int, C.c_int, C.c_int, i32p, i32p]
        L.kara_oracle_compress_window.restype = C.c_int
        L.kara_oracle_compress_window.argtypes = [
            C.POINTER(Layout), u16p, u16p, C.c_int, C.c_int, C.c_int, i32p, C.c_int, i32p, i32p,
            u16p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, C.c_int, C.c_int,
            i32p, i32p, f32p, f32p, i32p, i32p]
        L.kara_oracle_compress_windows.restype = C.c_int
        L.kara_oracle_compress_windows.argtypes = [
            C.POINTER(Layout), u16p, u16p, C.c_int, C.c_int, C.c_int, i32p, C.c_int, i32p, i32p, C.c_int,
            u16p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, C.c_int, C.c_int,
            i32p, i32p, f32p, f32p, i32p, i32p]
        u8p = C.POINTER(C.c_uint8)
        L.kara_oracle_policy_step.restype = C.c_int
        L.kara_oracle_policy_step.argtypes = [C.c_int, C.c_int, C.c_int, i32p, i32p, i32p, u8p, i32p, i32p, i32p,
                                              C.c_int, C.c_int, C.c_int, i32p, i32p, i32p, i32p, i32p, i32p]
        L.kara_oracle_policy_commit.restype = C.c_int
        L.kara_oracle_policy_commit.argtypes = [C.c_int, i32p, C.c_int, i32p, i32p, i32p, C.c_int, C.c_int,
                                                i32p, i32p, i32p]
        L.kara_oracle_window_queries.restype = C.c_int
        L.kara_oracle_window_queries.argtypes = [u16p, u16p, i32p, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, u16p]
        _LIB = L
    return _LIB


def _p(a, ty):
    return None if a is None else a.ctypes.data_as(C.POINTER(ty))


def _chk(a, dtype, name):
    if a is None:
        return None
    if not isinstance(a, np.ndarray) or a.dtype != dtype or not a.flags["C_CONTIGUOUS"]:
        raise TypeError(f"{name}: need C-contiguous numpy {np.dtype(dtype).name}")
    return a


def budget(n: int, ratio: float) -> int:
    return int(lib().kara_oracle_budget(int(n), float(ratio)))


def scores(q_bits: np.ndarray, k_bits: np.ndarray, buffer_only_U: int | None = None):
    """q_bits uint16 [W, G, d] (bf16 bit patterns), k_bits uint16 [n, d] -> (A64 [n], A32 [n])."""
    q_bits = _chk(q_bits, np.uint16, "q_bits")
    k_bits = _chk(k_bits, np.uint16, "k_bits")
    W, G, d = q_bits.shape
    n, d2 = k_bits.shape
    assert d == d2
    A64 = np.empty(n, np.float64)
    A32 = np.empty(n, np.float32)
    if buffer_only_U is None:
        rc = lib().kara_oracle_scores(_p(q_bits, C.c_uint16), G * d, d, _p(k_bits, C.c_uint16), d,
                                      W, G, n, d, _p(A64, C.c_double), _p(A32, C.c_float))
    else:
        rc = lib().kara_oracle_scores_buffer_queries(
            _p(q_bits, C.c_uint16), G * d, d, _p(k_bits, C.c_uint16), d,
            W, int(buffer_only_U), G, n, d, _p(A64, C.c_double), _p(A32, C.c_float))
    if rc:
        raise ValueError(f"kara_oracle_scores rc={rc}")
    return A64, A32


def select(A32: np.ndarray, keep: int, alpha: int, gamma: int):
    """-> dict(I [k], chunks [P], F [keep], n_chunk_added) from fp32 scores (Eq. 5-8 + C.3)."""
    A32 = _chk(np.ascontiguousarray(A32, np.float32), np.float32, "A32")
    n = A32.shape[0]
    k = keep - alpha
    P = alpha // (gamma - 2) if gamma > 2 else 0
    I = np.full(max(k, 1), -1, np.int32)
    ch = np.full(max(P, 1), -1, np.int32)
    F = np.full(max(keep, 1), -1, np.int32)
    added = np.zeros(1, np.int32)
    rc = lib().kara_oracle_select(_p(A32, C.c_float), n, keep, alpha, gamma,
                                  _p(I, C.c_int32), _p(ch, C.c_int32), _p(F, C.c_int32),
                                  _p(added, C.c_int32))
    if rc:
        raise ValueError(f"kara_oracle_select rc={rc}")
    return {"I": I[:k], "chunks": ch[:P], "F": F[:keep], "n_chunk_added": int(added[0])}


def compact_rows(old_rows: np.ndarray, h: int, W: int, U: int, t: int, F: np.ndarray):
    old_rows = _chk(old_rows, np.uint16, "old_rows")
    F = _chk(np.ascontiguousarray(F, np.int32), np.int32, "F")
    d = old_rows.shape[1]
    assert old_rows.shape[0] == h + W + t
    keep = F.shape[0]
    new_rows = np.empty((h + keep + U + t, d), np.uint16)
    rc = lib().kara_oracle_compact_rows(_p(old_rows, C.c_uint16), h, W, U, t, d, _p(F, C.c_int32),
                                        keep, _p(new_rows, C.c_uint16))
    if rc:
        raise ValueError(f"kara_oracle_compact_rows rc={rc}")
    return new_rows


def metadata(block_table, seq_lens, win_start, block_size, W, U, keep, free_list, free_count):
    """In place on the int32 arrays; free_count is an int32 array of shape [1]."""
    block_table = _chk(block_table, np.int32, "block_table")
    n_seqs, max_blocks = block_table.shape
    rc = lib().kara_oracle_metadata(n_seqs, max_blocks, block_size, _p(block_table, C.c_int32),
                                    _p(_chk(seq_lens, np.int32, "seq_lens"), C.c_int32),
                                    _p(_chk(win_start, np.int32, "win_start"), C.c_int32),
                                    W, U, keep, _p(_chk(free_list, np.int32, "free_list"), C.c_int32),
                                    _p(_chk(free_count, np.int32, "free_count"), C.c_int32))
    if rc:
        raise ValueError(f"kara_oracle_metadata rc={rc}")


def compress_window(layout: Layout, k_pool, v_pool, layer_begin, layer_end, block_table, seq_lens,
                    win_start, window_q, n_q_heads, W, U, ratio, alpha, gamma, commit,
                    free_list, free_count, scores_in=None, want_debug=True, n_windows=1):
    """Whole path O1-O11 on host images (all modified in place).  Returns dict of debug dumps.
    n_windows > 1: prefill, kara_oracle_compress_windows (dumps get a window axis after the sequence axis).

    k_pool / v_pool: uint16 numpy (bf16 bits), any shape, addressed through `layout` strides.
    window_q: uint16 [layers, n_seqs, W, n_q_heads, d] or None when scores_in is given.
    """
    k_pool = _chk(k_pool, np.uint16, "k_pool")
    v_pool = _chk(v_pool, np.uint16, "v_pool")
    block_table = _chk(block_table, np.int32, "block_table")
    seq_lens = _chk(seq_lens, np.int32, "seq_lens")
    win_start = _chk(win_start, np.int32, "win_start")
    window_q = _chk(window_q, np.uint16, "window_q")
    scores_in = _chk(scores_in, np.float32, "scores_in")
    free_list = _chk(free_list, np.int32, "free_list")
    free_count = _chk(free_count, np.int32, "free_count")
    n_seqs, max_blocks = block_table.shape
    nL = layer_end - layer_begin
    n = W - U
    keep = budget(n, ratio)
    k = keep - alpha
    units = nL * n_seqs * layout.n_kv_heads
    out = {"keep": keep, "k": k}
    s_out = i_out = f_out = None
    NW = int(n_windows)
    lead = (nL, n_seqs) if NW == 1 else (nL, n_seqs, NW)
    if want_debug:
        s_out = np.zeros(lead + (layout.n_kv_heads, n), np.float32)
        i_out = np.full(lead + (layout.n_kv_heads, max(k, 1)), -1, np.int32)
        f_out = np.full(lead + (layout.n_kv_heads, max(keep, 1)), -1, np.int32)
    del units
    if NW > 1:
        rc = lib().kara_oracle_compress_windows(
            C.byref(layout), _p(k_pool, C.c_uint16), _p(v_pool, C.c_uint16), layer_begin, layer_end,
            n_seqs, _p(block_table, C.c_int32), max_blocks, _p(seq_lens, C.c_int32),
            _p(win_start, C.c_int32), NW, _p(window_q, C.c_uint16), n_q_heads, W, U, float(ratio),
            alpha, gamma, int(bool(commit)), _p(free_list, C.c_int32), _p(free_count, C.c_int32),
            _p(scores_in, C.c_float), _p(s_out, C.c_float), _p(i_out, C.c_int32), _p(f_out, C.c_int32))
        if rc:
            raise ValueError(f"kara_oracle_compress_windows rc={rc}")
        out.update(scores=s_out, idx_topk=i_out, idx_final=f_out)
        return out
    rc = lib().kara_oracle_compress_window(
        C.byref(layout), _p(k_pool, C.c_uint16), _p(v_pool, C.c_uint16), layer_begin, layer_end,
        n_seqs, _p(block_table, C.c_int32), max_blocks, _p(seq_lens, C.c_int32),
        _p(win_start, C.c_int32), _p(window_q, C.c_uint16), n_q_heads, W, U, float(ratio),
        alpha, gamma, int(bool(commit)), _p(free_list, C.c_int32), _p(free_count, C.c_int32),
        _p(scores_in, C.c_float), _p(s_out, C.c_float), _p(i_out, C.c_int32), _p(f_out, C.c_int32))
    if rc:
        raise ValueError(f"kara_oracle_compress_window rc={rc}")
    out.update(scores=s_out, idx_topk=i_out, idx_final=f_out)
    return out


def policy_step(block_table, seq_lens, uncompressed, active, free_list, free_count, step_counter, block_size,
                delta, W, max_select):
    """One decoding step of Alg. 1 (in place on the int32 arrays; step_counter / free_count are int32 [1]).
    Returns dict(sel_ids, sel_count, sel_block_table, sel_seq_lens, sel_win_start, exhausted)."""
    block_table = _chk(block_table, np.int32, "block_table")
    n_seqs, max_blocks = block_table.shape
    sel_ids = np.empty(max(max_select, 1), np.int32)
    sel_sl = np.empty(max(max_select, 1), np.int32)
    sel_ws = np.empty(max(max_select, 1), np.int32)
    sel_bt = np.empty((max(max_select, 1), max_blocks), np.int32)
    cnt = np.zeros(1, np.int32)
    exh = np.zeros(1, np.int32)
    act = None if active is None else _chk(active, np.uint8, "active")
    rc = lib().kara_oracle_policy_step(
        n_seqs, max_blocks, block_size, _p(block_table, C.c_int32), _p(_chk(seq_lens, np.int32, "seq_lens"), C.c_int32),
        _p(_chk(uncompressed, np.int32, "uncompressed"), C.c_int32), _p(act, C.c_uint8),
        _p(_chk(free_list, np.int32, "free_list"), C.c_int32), _p(_chk(free_count, np.int32, "free_count"), C.c_int32),
        _p(_chk(step_counter, np.int32, "step_counter"), C.c_int32), delta, W, max_select,
        _p(sel_ids, C.c_int32), _p(cnt, C.c_int32), _p(sel_bt, C.c_int32), _p(sel_sl, C.c_int32), _p(sel_ws, C.c_int32),
        _p(exh, C.c_int32))
    if rc:
        raise ValueError(f"kara_oracle_policy_step rc={rc}")
    return dict(sel_ids=sel_ids[:max_select], sel_count=int(cnt[0]), sel_block_table=sel_bt[:max_select],
                sel_seq_lens=sel_sl[:max_select], sel_win_start=sel_ws[:max_select], exhausted=int(exh[0]))


def policy_commit(sel, keep, U, block_table, seq_lens, uncompressed):
    """UpdateMetadata of the running queue after the selected sub-batch was compressed (in place)."""
    block_table = _chk(block_table, np.int32, "block_table")
    rc = lib().kara_oracle_policy_commit(
        block_table.shape[1], _p(np.ascontiguousarray(sel["sel_ids"], np.int32), C.c_int32), int(sel["sel_count"]),
        _p(np.ascontiguousarray(sel["sel_block_table"], np.int32), C.c_int32),
        _p(np.ascontiguousarray(sel["sel_seq_lens"], np.int32), C.c_int32),
        _p(np.ascontiguousarray(sel["sel_win_start"], np.int32), C.c_int32), keep, U, _p(block_table, C.c_int32),
        _p(_chk(seq_lens, np.int32, "seq_lens"), C.c_int32), _p(_chk(uncompressed, np.int32, "uncompressed"), C.c_int32))
    if rc:
        raise ValueError(f"kara_oracle_policy_commit rc={rc}")


def window_queries(hidden_bits, wq_bits, positions, rope_theta, n_q_heads, d):
    """hidden uint16 [T, Dm], wq uint16 [Hq*d, Dm] (bf16 bits), positions int32 [T] or None -> uint16 [T, Hq, d]."""
    hidden_bits = _chk(hidden_bits, np.uint16, "hidden")
    wq_bits = _chk(wq_bits, np.uint16, "wq")
    T, Dm = hidden_bits.shape
    assert wq_bits.shape == (n_q_heads * d, Dm)
    pos = None if positions is None else _chk(np.ascontiguousarray(positions, np.int32), np.int32, "positions")
    out = np.empty((T, n_q_heads, d), np.uint16)
    rc = lib().kara_oracle_window_queries(_p(hidden_bits, C.c_uint16), _p(wq_bits, C.c_uint16), _p(pos, C.c_int32),
                                          float(rope_theta), T, Dm, n_q_heads, d, _p(out, C.c_uint16))
    if rc:
        raise ValueError(f"kara_oracle_window_queries rc={rc}")
    return out
