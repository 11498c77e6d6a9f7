"""Thin ctypes binding of libkara.so (include/kara.h) — argument marshalling only.

Same names as the C ABI: kara_init_cache, kara_attach_pool, kara_compress_window,
kara_compress_window_host, kara_gather_debug, ...  Every step of the method runs in the CUDA
kernels behind the ABI; torch is used for device memory and streams.  There is no CPU
fallback: if libkara.so is missing or a call fails, a KaraError is raised.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np
import torch

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "libkara.so"
_LIB = None

KARA_OK, KARA_EINVAL, KARA_EBUDGET, KARA_EUNSUPPORTED, KARA_ECUDA, KARA_ENOMEM = 0, -1, -2, -3, -4, -5
KARA_COMMIT, KARA_KEEP_DEBUG, KARA_SCORE_QBUF_ONLY, KARA_SCORE_SIMT = 1, 2, 4, 8
(KARA_DBG_K_LOGICAL, KARA_DBG_V_LOGICAL, KARA_DBG_SCORES, KARA_DBG_IDX_TOPK, KARA_DBG_IDX_FINAL,
 KARA_DBG_BLOCK_TABLE_ROW, KARA_DBG_FREE_LIST) = range(7)
KARA_ST_BAD_BLOCK, KARA_ST_SHORT_SEQ, KARA_ST_TABLE_OVERFLOW, KARA_ST_FREE_OVERFLOW = 1, 2, 4, 8
KARA_STATIC_SCRATCH_BYTES = 1048576

# every symbol include/kara.h declares: (restype, argtypes)
_vp, _i, _i64, _sz, _d, _u = C.c_void_p, C.c_int, C.c_int64, C.c_size_t, C.c_double, C.c_uint
SYMBOLS = {
    "kara_init_cache": (_vp, [_i, _i, _i, _i]),
    "kara_destroy": (None, [_vp]),
    "kara_pool_bytes": (_i64, [_vp, _i64]),
    "kara_block_bytes": (_i64, [_vp]),
    "kara_attach_pool": (_i, [_vp, _vp, _vp, _i64, _vp, _vp]),
    "kara_budget": (_i, [_i, _d]),
    "kara_workspace_bytes": (_sz, [_vp, _i, _i, _i, _i, _i, _d, _i]),
    "kara_compress_window": (_i, [_vp, _i, _i, _i, _vp, _i, _vp, _vp, _vp, _i, _i, _i, _d, _i, _i, _u,
                                  _vp, _sz, _vp]),
    "kara_compress_windows": (_i, [_vp, _i, _i, _i, _vp, _i, _vp, _vp, _i, _vp, _i, _i, _i, _d, _i, _i, _u,
                                   _vp, _sz, _vp]),
    "kara_compress_window_host": (_i, [_vp, _i, _i, _i, _vp, _i, _vp, _vp, _vp, _i, _i, _i, _d, _i, _i,
                                       _u, _vp, _vp]),
    "kara_policy_step": (_i, [_vp, _i, _vp, _i, _vp, _vp, _vp, _vp, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "kara_policy_commit": (_i, [_vp, _i, _vp, _vp, _vp, _vp, _vp, _i, _i, _d, _vp, _i, _vp, _vp, _vp]),
    "kara_window_queries_workspace_bytes": (_sz, [_i, _i]),
    "kara_window_queries": (_i, [_vp, _vp, _vp, _i, _d, _i, _i, _i, _i, _vp, _vp, _sz, _vp]),
    "kara_window_queries_static": (_i, [_vp, _vp, _vp, _i, _d, _i, _i, _i, _i, _vp, _vp]),
    "kara_gather_debug": (_i, [_vp, _i, _i, _i, _i, _vp, _vp, _i, _vp, _i64, C.POINTER(_i64)]),
    "kara_status": (_i, [_vp, C.POINTER(C.c_int32)]),
    "kara_last_launch_count": (_i, [_vp]),
    "kara_last_score_path": (_i, [_vp]),
    "kara_last_score_path_reason": (C.c_char_p, [_vp]),
    "kara_enable_score_timing": (_i, [_vp, _i]),
    "kara_score_kernel_ms": (C.c_float, [_vp]),
    "kara_last_error": (C.c_char_p, []),
}


class KaraError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libkara error {code}: {msg}")
        self.code = code


def lib() -> C.CDLL:
    """Load libkara.so (built by paper_2607_01237_b200.build).  Fails loudly if it is missing."""
    global _LIB
    if _LIB is None:
        if not _SO.exists():
            raise KaraError(KARA_EINVAL, f"{_SO} not built — run `python -m paper_2607_01237_b200.build` "
                                         "(there is no CPU fallback)")
        L = C.CDLL(str(_SO))
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _LIB = L
    return _LIB


def _check(rc: int) -> None:
    if rc != KARA_OK:
        raise KaraError(rc, lib().kara_last_error().decode())


def _ptr(t: torch.Tensor | None) -> int | None:
    return None if t is None else t.data_ptr()


def kara_budget(n: int, ratio: float) -> int:
    return int(lib().kara_budget(int(n), float(ratio)))


def kara_window_queries(hidden: torch.Tensor, wq: torch.Tensor, positions: torch.Tensor | None, rope_theta: float,
                        n_q_heads: int, head_dim: int, out: torch.Tensor | None = None, max_position: int | None = None,
                        stream: torch.cuda.Stream | None = None) -> torch.Tensor:
    """kara_window_queries: hidden [T, Dm] bf16, wq [Hq*d, Dm] bf16, positions int32 [T] or None -> [T, Hq, d] bf16."""
    T, Dm = hidden.shape
    assert hidden.is_cuda and hidden.is_contiguous() and hidden.dtype == torch.bfloat16
    assert wq.shape == (n_q_heads * head_dim, Dm) and wq.is_contiguous() and wq.dtype == torch.bfloat16
    if out is None:
        out = torch.empty(T, n_q_heads, head_dim, dtype=torch.bfloat16, device=hidden.device)
    assert out.is_contiguous() and out.dtype == torch.bfloat16 and out.numel() == T * n_q_heads * head_dim
    ws = None
    if positions is not None:
        assert positions.dtype == torch.int32 and positions.is_cuda and positions.numel() == T
        if max_position is None:
            max_position = int(positions.max()) if T else 0
        ws = torch.empty(max(int(lib().kara_window_queries_workspace_bytes(max_position, head_dim)), 16), dtype=torch.uint8,
                         device=hidden.device)
    st = (stream or torch.cuda.current_stream(hidden.device)).cuda_stream
    _check(lib().kara_window_queries(_ptr(hidden), _ptr(wq), _ptr(positions), max_position or 0, float(rope_theta), T, Dm,
                                     n_q_heads, head_dim, _ptr(out), _ptr(ws), ws.numel() if ws is not None else 0, st))
    return out


def kara_window_queries_static(hidden: torch.Tensor, wq: torch.Tensor, positions: torch.Tensor | None, rope_theta: float,
                               n_q_heads: int, head_dim: int, out: torch.Tensor, max_position: int,
                               stream: torch.cuda.Stream | None = None) -> torch.Tensor:
    """kara_window_queries_static: kara_window_queries without a workspace, for callers that must not allocate device memory
    during decoding (the rotary tables go into libkara's built-in 1 MiB device array; see include/kara.h for the limit on
    max_position, the first-call set-up and why calls on one GPU must not overlap).  This binding allocates nothing either:
    `out` [T, Hq, d] bf16 and `max_position` are the caller's, nothing is read back from the device."""
    T, Dm = hidden.shape
    assert hidden.is_cuda and hidden.is_contiguous() and hidden.dtype == torch.bfloat16
    assert wq.shape == (n_q_heads * head_dim, Dm) and wq.is_contiguous() and wq.dtype == torch.bfloat16
    assert out.is_cuda and out.is_contiguous() and out.dtype == torch.bfloat16 and out.numel() == T * n_q_heads * head_dim
    if positions is not None:
        assert positions.dtype == torch.int32 and positions.is_cuda and positions.numel() == T
    st = (stream or torch.cuda.current_stream(hidden.device)).cuda_stream
    _check(lib().kara_window_queries_static(_ptr(hidden), _ptr(wq), _ptr(positions), int(max_position), float(rope_theta), T,
                                            Dm, n_q_heads, head_dim, _ptr(out), st))
    return out


class KaraCache:
    """Handle of kara_init_cache + kara_attach_pool over caller-owned torch tensors."""

    def __init__(self, block_size: int, n_layers: int, n_kv_heads: int, head_dim: int):
        self.block_size, self.n_layers, self.n_kv_heads, self.head_dim = block_size, n_layers, n_kv_heads, head_dim
        self._h = lib().kara_init_cache(block_size, n_layers, n_kv_heads, head_dim)
        if not self._h:
            raise KaraError(KARA_EUNSUPPORTED, lib().kara_last_error().decode())
        self._keep = []          # tensors the library points into
        self._workspace = None

    def close(self):
        if getattr(self, "_h", None):
            lib().kara_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- kara_pool_bytes / kara_block_bytes ---------------------------------------------------
    def pool_bytes(self, num_blocks: int) -> int:
        return int(lib().kara_pool_bytes(self._h, num_blocks))

    def block_bytes(self) -> int:
        return int(lib().kara_block_bytes(self._h))

    # -- kara_attach_pool ------------------------------------------------------------------------
    def attach_pool(self, k_pool: torch.Tensor, v_pool: torch.Tensor, free_list: torch.Tensor,
                    free_count: torch.Tensor) -> None:
        L, NB, Hkv, bs, d = k_pool.shape
        assert (L, Hkv, bs, d) == (self.n_layers, self.n_kv_heads, self.block_size, self.head_dim)
        assert k_pool.is_cuda and k_pool.is_contiguous() and k_pool.dtype == torch.bfloat16
        assert v_pool.shape == k_pool.shape and v_pool.is_contiguous() and v_pool.dtype == torch.bfloat16
        assert free_list.dtype == torch.int32 and free_list.numel() >= NB and free_count.dtype == torch.int32
        self.num_blocks = NB
        self._keep = [k_pool, v_pool, free_list, free_count]
        _check(lib().kara_attach_pool(self._h, _ptr(k_pool), _ptr(v_pool), NB, _ptr(free_list), _ptr(free_count)))

    # -- kara_workspace_bytes ----------------------------------------------------------------------
    def workspace_bytes(self, n_layers_in_call, n_seqs, n_q_heads, W, U, ratio, alpha) -> int:
        return int(lib().kara_workspace_bytes(self._h, n_layers_in_call, n_seqs, n_q_heads, W, U, float(ratio), alpha))

    def _get_workspace(self, nbytes: int, device) -> torch.Tensor:
        if self._workspace is None or self._workspace.numel() < nbytes or self._workspace.device != device:
            self._workspace = torch.empty(nbytes, dtype=torch.uint8, device=device)
        return self._workspace

    # -- kara_compress_window ------------------------------------------------------------------------
    def compress_window(self, layer_begin: int, layer_end: int, block_table: torch.Tensor,
                        seq_lens: torch.Tensor, win_start: torch.Tensor | None, window_q: torch.Tensor,
                        W: int, U: int, ratio: float, alpha: int, gamma: int, flags: int = KARA_COMMIT,
                        workspace: torch.Tensor | None = None, stream: torch.cuda.Stream | None = None) -> None:
        n_seqs, max_blocks = block_table.shape
        nL, S, Wq, Hq, d = window_q.shape
        assert (nL, S, Wq, d) == (layer_end - layer_begin, n_seqs, W, self.head_dim), "window_q shape"
        assert window_q.is_cuda and window_q.is_contiguous() and window_q.dtype == torch.bfloat16
        assert block_table.dtype == torch.int32 and block_table.is_contiguous() and block_table.is_cuda
        assert seq_lens.dtype == torch.int32 and seq_lens.is_cuda
        if workspace is None:
            workspace = self._get_workspace(self.workspace_bytes(nL, n_seqs, Hq, W, U, ratio, alpha), window_q.device)
        st = (stream or torch.cuda.current_stream(window_q.device)).cuda_stream
        _check(lib().kara_compress_window(self._h, layer_begin, layer_end, n_seqs, _ptr(block_table), max_blocks,
                                          _ptr(seq_lens), _ptr(win_start), _ptr(window_q), Hq, W, U, float(ratio),
                                          alpha, gamma, flags, _ptr(workspace), workspace.numel(), st))

    # -- kara_compress_windows (prefill: n_windows disjoint windows per sequence) ---------------------------
    def compress_windows(self, layer_begin: int, layer_end: int, block_table: torch.Tensor, seq_lens: torch.Tensor,
                         win_start: torch.Tensor | None, n_windows: int, window_q: torch.Tensor, W: int, U: int,
                         ratio: float, alpha: int, gamma: int, flags: int = KARA_COMMIT,
                         workspace: torch.Tensor | None = None, stream: torch.cuda.Stream | None = None) -> None:
        n_seqs, max_blocks = block_table.shape
        nL, S, Wq, Hq, d = window_q.shape
        assert (nL, S, Wq, d) == (layer_end - layer_begin, n_seqs, n_windows * W, self.head_dim), "window_q shape"
        assert window_q.is_cuda and window_q.is_contiguous() and window_q.dtype == torch.bfloat16
        assert block_table.dtype == torch.int32 and block_table.is_contiguous() and block_table.is_cuda
        assert seq_lens.dtype == torch.int32 and seq_lens.is_cuda
        if workspace is None:
            workspace = self._get_workspace(self.workspace_bytes(nL, n_seqs * n_windows, Hq, W, U, ratio, alpha),
                                            window_q.device)
        st = (stream or torch.cuda.current_stream(window_q.device)).cuda_stream
        _check(lib().kara_compress_windows(self._h, layer_begin, layer_end, n_seqs, _ptr(block_table), max_blocks,
                                           _ptr(seq_lens), _ptr(win_start), n_windows, _ptr(window_q), Hq, W, U,
                                           float(ratio), alpha, gamma, flags, _ptr(workspace), workspace.numel(), st))

    # -- kara_compress_window_host -------------------------------------------------------------------
    def compress_window_host(self, layer_begin: int, layer_end: int, block_table: torch.Tensor,
                             seq_lens: torch.Tensor, win_start: torch.Tensor | None, window_q: torch.Tensor,
                             W: int, U: int, ratio: float, alpha: int, gamma: int, flags: int = KARA_COMMIT,
                             stream: torch.cuda.Stream | None = None) -> int:
        """Host (ideally pinned) tensors in, updated in place; returns the new free-block count."""
        n_seqs, max_blocks = block_table.shape
        nL, S, Wq, Hq, d = window_q.shape
        assert (nL, S, Wq, d) == (layer_end - layer_begin, n_seqs, W, self.head_dim), "window_q shape"
        for t in (block_table, seq_lens, window_q) + ((win_start,) if win_start is not None else ()):
            assert not t.is_cuda and t.is_contiguous()
        fc = torch.zeros(1, dtype=torch.int32).pin_memory()
        st = (stream or torch.cuda.current_stream()).cuda_stream
        _check(lib().kara_compress_window_host(self._h, layer_begin, layer_end, n_seqs, _ptr(block_table), max_blocks,
                                               _ptr(seq_lens), _ptr(win_start), _ptr(window_q), Hq, W, U,
                                               float(ratio), alpha, gamma, flags, _ptr(fc), st))
        return int(fc[0])

    # -- kara_policy_step / kara_policy_commit (Alg. 1 on the device) -----------------------------------------
    def policy_step(self, block_table, seq_lens, uncompressed, active, step_counter, delta, W, sel, exhausted,
                    stream: torch.cuda.Stream | None = None) -> None:
        """`sel` = dict of device tensors ids [m], count [1], block_table [m, max_blocks], seq_lens [m], win_start [m]."""
        n_seqs, max_blocks = block_table.shape
        m = sel["ids"].numel()
        assert sel["block_table"].shape == (m, max_blocks) and sel["block_table"].is_contiguous()
        for x in (block_table, seq_lens, uncompressed, step_counter, exhausted, *sel.values()):
            assert x.is_cuda and x.dtype == torch.int32 and x.is_contiguous()
        assert active is None or (active.is_cuda and active.dtype == torch.uint8)
        st = (stream or torch.cuda.current_stream(block_table.device)).cuda_stream
        _check(lib().kara_policy_step(self._h, n_seqs, _ptr(block_table), max_blocks, _ptr(seq_lens), _ptr(uncompressed),
                                      _ptr(active), _ptr(step_counter), delta, W, m, _ptr(sel["ids"]), _ptr(sel["count"]),
                                      _ptr(sel["block_table"]), _ptr(sel["seq_lens"]), _ptr(sel["win_start"]),
                                      _ptr(exhausted), st))

    def policy_commit(self, sel, W, U, ratio, block_table, seq_lens, uncompressed,
                      stream: torch.cuda.Stream | None = None) -> None:
        m = sel["ids"].numel()
        st = (stream or torch.cuda.current_stream(block_table.device)).cuda_stream
        _check(lib().kara_policy_commit(self._h, m, _ptr(sel["ids"]), _ptr(sel["count"]), _ptr(sel["block_table"]),
                                        _ptr(sel["seq_lens"]), _ptr(sel["win_start"]), W, U, float(ratio),
                                        _ptr(block_table), block_table.shape[1], _ptr(seq_lens), _ptr(uncompressed), st))

    # -- kara_gather_debug -----------------------------------------------------------------------------
    def gather_debug(self, what: int, layer: int, seq: int, kv_head: int, block_table: torch.Tensor | None = None,
                     seq_lens: torch.Tensor | None = None) -> np.ndarray:
        max_blocks = block_table.shape[1] if block_table is not None else 0
        if what in (KARA_DBG_K_LOGICAL, KARA_DBG_V_LOGICAL):
            cap = int(seq_lens[seq]) * self.head_dim * 2
            out = np.empty(max(cap // 2, 1), np.uint16)
        elif what == KARA_DBG_SCORES:
            out = np.empty(4096, np.float32)
        else:
            out = np.empty(max(self.num_blocks, max_blocks, 4096), np.int32)
        cnt = C.c_int64(0)
        _check(lib().kara_gather_debug(self._h, what, layer, seq, kv_head, _ptr(block_table), _ptr(seq_lens),
                                       max_blocks, out.ctypes.data, out.nbytes, C.byref(cnt)))
        out = out[: cnt.value]
        if what in (KARA_DBG_K_LOGICAL, KARA_DBG_V_LOGICAL):
            out = out.reshape(-1, self.head_dim)
        return out

    # -- kara_status and friends ------------------------------------------------------------------------
    def status(self) -> int:
        s = C.c_int32(0)
        _check(lib().kara_status(self._h, C.byref(s)))
        return int(s.value)

    def last_launch_count(self) -> int:
        return int(lib().kara_last_launch_count(self._h))

    def last_score_path(self) -> int:
        return int(lib().kara_last_score_path(self._h))

    def last_score_path_reason(self) -> str:
        return lib().kara_last_score_path_reason(self._h).decode()

    def enable_score_timing(self, enable: bool = True) -> None:
        _check(lib().kara_enable_score_timing(self._h, int(enable)))

    def score_kernel_ms(self) -> float:
        return float(lib().kara_score_kernel_ms(self._h))
