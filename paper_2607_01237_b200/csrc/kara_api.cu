// kara_api.cu — the C ABI of include/kara.h: argument checking, workspace carving, launch order.
// No step of the method runs on the host: a1 = score kernel, a2-a4 = select_compact kernel,
// a5 = metadata kernel, all on the caller's stream with no host synchronisation in between.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include "kara_internal.h"
#include "score_tc.h"

using namespace kara;

// The device status words (include/kara.h, kara_status) live in the library's own device image, one 32-byte slot per live
// handle, NOT in the caller's workspace: a workspace may be freed and handed out again at the same address with garbage in
// it, or be shared by two handles, and neither may turn into fault bits or erase another handle's.  No allocation: the
// array is part of every GPU's copy of the module; a handle looks its slot's address up when a pool is attached.
constexpr int kMaxHandles = 4096;
static __device__ __align__(32) int32_t g_status_slots[kMaxHandles][8];

struct kara_cache {
  Geom g{};
  void* k_pool = nullptr;
  void* v_pool = nullptr;
  int32_t* free_list = nullptr;
  int32_t* free_count = nullptr;
  bool attached = false;
  // last call (for kara_gather_debug / kara_status)
  bool have_last = false;
  Call last{};
  int last_launches = 0;
  int last_score_path = 0;
  const char* last_score_reason = "";   // why the CUDA-core kernel ran ("" when the tcgen05 kernel did)
  // sticky device status word: g_status_slots[status_slot] on the device of the attached pool (see kara_status)
  int status_slot = -1;
  int32_t* status_dev = nullptr;
  // score-kernel timing
  bool timing = false;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  bool ev_recorded = false;
  // staging owned by kara_compress_window_host
  void* d_q = nullptr; size_t d_q_bytes = 0;
  int32_t* d_bt = nullptr; size_t d_bt_bytes = 0;
  int32_t* d_sl = nullptr; int32_t* d_ws = nullptr; size_t d_sl_bytes = 0;
  void* d_work = nullptr; size_t d_work_bytes = 0;
  ScoreTcState tc{};
};

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return code;
}
#define KARA_CUDA(expr)                                                                  \
  do {                                                                                   \
    cudaError_t e__ = (expr);                                                            \
    if (e__ != cudaSuccess) return fail(KARA_ECUDA, "%s: %s", #expr, cudaGetErrorString(e__)); \
  } while (0)

std::mutex g_slot_mutex;
bool g_slot_used[kMaxHandles] = {};

int take_status_slot() {
  std::lock_guard<std::mutex> lock(g_slot_mutex);
  for (int i = 0; i < kMaxHandles; ++i)
    if (!g_slot_used[i]) { g_slot_used[i] = true; return i; }
  return -1;
}
void release_status_slot(int i) {
  if (i < 0) return;
  std::lock_guard<std::mutex> lock(g_slot_mutex);
  g_slot_used[i] = false;
}

int ilog2_exact(int x) {
  int l = 0;
  while ((1 << l) < x) ++l;
  return (1 << l) == x ? l : -1;
}

int budget(int n, double ratio) {
  if (n <= 0 || !(ratio > 0.0) || ratio > 1.0) return -1;
  return (int)std::ceil(ratio * (double)n - 1e-9);   // reading G5
}

// KARA_SCORE_QBUF_ONLY packs the U buffer tokens of 2^x query heads into one 128-row tile: tokens per tile = the largest
// power of two <= min(U, 128), heads per tile = 128 / that.
void qbuf_tiling(int U, int* tile_toks, int* hpt_log2) {
  int tt = 1, l = 0;
  while (tt * 2 <= U && tt * 2 <= 128) tt *= 2;
  while ((tt << l) < 128) ++l;
  *tile_toks = tt;
  *hpt_log2 = l;
}

// Query tiles per unit of the two score variants: full window (128 rows x one head) and, if U > 0, buffer queries only.
// The packed variant can have MORE tiles per unit than the full one (W = 100, U = 65, G = 3: 2 token tiles x 2 head
// tiles = 4 against 3), so the workspace reserves strips for whichever needs more and serves either flag.
void tiles_per_unit(int W, int U, int G, int* full, int* qbuf) {
  *full = (W + 127) / 128 * G;
  *qbuf = 0;
  if (U > 0) {
    int tt, l;
    qbuf_tiling(U, &tt, &l);
    *qbuf = (U + tt - 1) / tt * ((G + (1 << l) - 1) >> l);
  }
}

WsLayout ws_layout(int units, int n, int k, int keep, int tpu_full, int tpu_qbuf) {
  WsLayout w{};
  w.parts = strips_bound(units, tpu_full);
  if (tpu_qbuf > 0 && strips_bound(units, tpu_qbuf) > w.parts) w.parts = strips_bound(units, tpu_qbuf);
  w.n_pad = round_up(n, 4);
  w.k_pad = round_up(k > 0 ? k : 1, 4);
  w.keep_pad = round_up(keep > 0 ? keep : 1, 4);
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += (bytes + 255) / 256 * 256; return o; };
  w.status_off = take(8 * sizeof(int32_t));
  w.partial_off = take(sizeof(float) * (size_t)units * w.parts * w.n_pad);
  w.scores_off = take(sizeof(float) * (size_t)units * w.n_pad);
  w.topk_off = take(sizeof(int32_t) * (size_t)units * w.k_pad);
  w.final_off = take(sizeof(int32_t) * (size_t)units * w.keep_pad);
  w.total = off;
  return w;
}

int check_geometry(const kara_cache* c, int layer_begin, int layer_end, int n_seqs, int n_q_heads, int W,
                   int U, double ratio, int alpha, int gamma, int* keep_out) {
  if (!c) return fail(KARA_EINVAL, "null handle");
  if (layer_begin < 0 || layer_end > c->g.n_layers || layer_begin >= layer_end)
    return fail(KARA_EINVAL, "layer range [%d,%d) outside [0,%d)", layer_begin, layer_end, c->g.n_layers);
  if (n_seqs <= 0) return fail(KARA_EINVAL, "n_seqs=%d", n_seqs);
  if (n_q_heads <= 0 || n_q_heads % c->g.n_kv_heads != 0)
    return fail(KARA_EINVAL, "n_q_heads=%d not a multiple of n_kv_heads=%d", n_q_heads, c->g.n_kv_heads);
  if (U < 0 || W <= U) return fail(KARA_EINVAL, "need 0 <= U < W (W=%d U=%d)", W, U);
  const int n = W - U;
  if (n > kMaxN) return fail(KARA_EUNSUPPORTED, "n = W-U = %d exceeds %d", n, kMaxN);
  const int keep = budget(n, ratio);
  if (keep < 0) return fail(KARA_EINVAL, "ratio=%g outside (0,1]", ratio);
  if (alpha < 0) return fail(KARA_EINVAL, "alpha=%d", alpha);
  if (gamma < 3) return fail(KARA_EBUDGET, "gamma=%d < 3 (PAPER.md:L140)", gamma);
  if (keep - alpha < 1) return fail(KARA_EBUDGET, "keep-alpha = %d-%d < 1", keep, alpha);
  if (keep > n) return fail(KARA_EBUDGET, "keep=%d > n=%d", keep, n);
  *keep_out = keep;
  return KARA_OK;
}

}  // namespace

// kara_last_error's message, for the translation units that hold an ABI entry point of their own
int kara::api_fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return code;
}

extern "C" {

const char* kara_last_error(void) { return g_err; }

int kara_budget(int n, double ratio) { return budget(n, ratio); }

kara_cache* kara_init_cache(int block_size, int n_layers, int n_kv_heads, int head_dim) {
  const int l2 = ilog2_exact(block_size);
  if (l2 < 0 || block_size < 16 || block_size > 256) {
    fail(KARA_EUNSUPPORTED, "block_size=%d: need a power of two in [16,256]", block_size);
    return nullptr;
  }
  if (head_dim != 64 && head_dim != 128) {
    fail(KARA_EUNSUPPORTED, "head_dim=%d: need 64 or 128", head_dim);
    return nullptr;
  }
  if (n_layers <= 0 || n_kv_heads <= 0) {
    fail(KARA_EINVAL, "n_layers=%d n_kv_heads=%d", n_layers, n_kv_heads);
    return nullptr;
  }
  kara_cache* c = new (std::nothrow) kara_cache();
  if (!c) { fail(KARA_ENOMEM, "host allocation failed"); return nullptr; }
  c->status_slot = take_status_slot();
  if (c->status_slot < 0) {
    delete c;
    fail(KARA_ENOMEM, "more than %d live handles (kara_destroy the ones no longer used)", kMaxHandles);
    return nullptr;
  }
  c->g.bs = block_size;
  c->g.bs_log2 = l2;
  c->g.n_layers = n_layers;
  c->g.n_kv_heads = n_kv_heads;
  c->g.d = head_dim;
  c->g.sH = (long long)block_size * head_dim;
  c->g.sB = c->g.sH * n_kv_heads;
  return c;
}

void kara_destroy(kara_cache* c) {
  if (!c) return;
  if (c->ev0) cudaEventDestroy(c->ev0);
  if (c->ev1) cudaEventDestroy(c->ev1);
  if (c->d_q) cudaFree(c->d_q);
  if (c->d_bt) cudaFree(c->d_bt);
  if (c->d_sl) cudaFree(c->d_sl);
  if (c->d_ws) cudaFree(c->d_ws);
  if (c->d_work) cudaFree(c->d_work);
  release_status_slot(c->status_slot);
  delete c;
}

int64_t kara_block_bytes(const kara_cache* c) {
  return c ? (int64_t)c->g.sB * 2 * c->g.n_layers : KARA_EINVAL;
}

int64_t kara_pool_bytes(const kara_cache* c, int64_t num_blocks) {
  if (!c || num_blocks <= 0) return KARA_EINVAL;
  return (int64_t)c->g.n_layers * num_blocks * c->g.sB * 2;
}

int kara_attach_pool(kara_cache* c, void* k_pool, void* v_pool, int64_t num_blocks, int32_t* free_list,
                     int32_t* free_count) {
  if (!c || !k_pool || !v_pool || !free_list || !free_count || num_blocks <= 0)
    return fail(KARA_EINVAL, "kara_attach_pool: null pointer or num_blocks=%lld", (long long)num_blocks);
  if (((uintptr_t)k_pool | (uintptr_t)v_pool) & 255u)
    return fail(KARA_EINVAL, "pools must be 256-byte aligned");
  c->k_pool = k_pool;
  c->v_pool = v_pool;
  c->free_list = free_list;
  c->free_count = free_count;
  c->g.num_blocks = num_blocks;
  c->g.sL = c->g.sB * num_blocks;
  c->have_last = false;
  // this handle's status slot on the current device (the pool's), cleared: a destroyed handle may have left bits in it
  void* slots = nullptr;
  KARA_CUDA(cudaGetSymbolAddress(&slots, g_status_slots));
  c->status_dev = static_cast<int32_t*>(slots) + (size_t)c->status_slot * 8;
  KARA_CUDA(cudaMemset(c->status_dev, 0, 8 * sizeof(int32_t)));
  c->attached = true;
  int rc = score_tc_attach(&c->tc, c->g, k_pool);
  if (rc != KARA_OK) return fail(rc, "TMA descriptor for the K pool: %s", score_tc_error());
  return KARA_OK;
}

size_t kara_workspace_bytes(const kara_cache* c, int n_layers_in_call, int n_seqs, int n_q_heads, int W, int U,
                            double ratio, int alpha) {
  if (!c || n_layers_in_call <= 0 || n_seqs <= 0 || U < 0 || W <= U || n_q_heads <= 0 ||
      n_q_heads % c->g.n_kv_heads != 0)
    return 0;
  const int n = W - U;
  const int keep = budget(n, ratio);
  if (keep < 0) return 0;
  const int units = n_layers_in_call * n_seqs * c->g.n_kv_heads;
  int tpu_full, tpu_qbuf;
  tiles_per_unit(W, U, n_q_heads / c->g.n_kv_heads, &tpu_full, &tpu_qbuf);
  return ws_layout(units, n, keep - alpha, keep, tpu_full, tpu_qbuf).total;
}

int kara_compress_window(kara_cache* c, int layer_begin, int layer_end, int n_seqs, int32_t* block_table,
                         int max_blocks, int32_t* seq_lens, const int32_t* win_start, const void* window_q,
                         int n_q_heads, int W, int U, double ratio, int alpha, int gamma, unsigned flags,
                         void* workspace, size_t workspace_bytes, void* stream) {
  return kara_compress_windows(c, layer_begin, layer_end, n_seqs, block_table, max_blocks, seq_lens, win_start, 1,
                               window_q, n_q_heads, W, U, ratio, alpha, gamma, flags, workspace, workspace_bytes, stream);
}

int kara_compress_windows(kara_cache* c, int layer_begin, int layer_end, int n_seqs, int32_t* block_table,
                          int max_blocks, int32_t* seq_lens, const int32_t* win_start, int n_windows,
                          const void* window_q, int n_q_heads, int W, int U, double ratio, int alpha, int gamma,
                          unsigned flags, void* workspace, size_t workspace_bytes, void* stream) {
  int keep = 0;
  if (n_windows < 1) return fail(KARA_EINVAL, "n_windows=%d", n_windows);
  int rc = check_geometry(c, layer_begin, layer_end, n_seqs, n_q_heads, W, U, ratio, alpha, gamma, &keep);
  if (rc != KARA_OK) return rc;
  if (!c->attached) return fail(KARA_EINVAL, "kara_attach_pool has not been called");
  if (!block_table || !seq_lens || !window_q || !workspace || max_blocks <= 0)
    return fail(KARA_EINVAL, "null pointer argument or max_blocks=%d", max_blocks);
  if (((uintptr_t)window_q & 15u) || ((uintptr_t)workspace & 255u))
    return fail(KARA_EINVAL, "window_q must be 16-byte and workspace 256-byte aligned");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);

  const int nL = layer_end - layer_begin;
  const int n = W - U;
  const int units = nL * n_seqs * n_windows * c->g.n_kv_heads;
  int tpu_full, tpu_qbuf;
  tiles_per_unit(W, U, n_q_heads / c->g.n_kv_heads, &tpu_full, &tpu_qbuf);
  const WsLayout w = ws_layout(units, n, keep - alpha, keep, tpu_full, tpu_qbuf);
  if (workspace_bytes < w.total)
    return fail(KARA_ENOMEM, "workspace %zu bytes < %zu needed", workspace_bytes, w.total);

  Call k{};
  k.g = c->g;
  k.k_pool = static_cast<const __nv_bfloat16*>(c->k_pool);
  k.v_pool = static_cast<const __nv_bfloat16*>(c->v_pool);
  k.layer_begin = layer_begin;
  k.n_layers = nL;
  k.n_seqs = n_seqs;
  k.n_windows = n_windows;
  k.max_blocks = max_blocks;
  k.n_q_heads = n_q_heads;
  k.G = n_q_heads / c->g.n_kv_heads;
  k.W = W; k.U = U; k.n = n; k.keep = keep; k.k = keep - alpha;
  k.P = alpha / (gamma - 2);
  k.alpha = alpha; k.gamma = gamma;
  k.q_row_begin = (flags & KARA_SCORE_QBUF_ONLY) ? W - U : 0;
  k.q_tile_toks = 128; k.q_hpt_log2 = 0;
  if (flags & KARA_SCORE_QBUF_ONLY) {
    qbuf_tiling(U, &k.q_tile_toks, &k.q_hpt_log2);
  }
  if ((flags & KARA_SCORE_QBUF_ONLY) && U == 0)
    return fail(KARA_EINVAL, "KARA_SCORE_QBUF_ONLY needs U > 0");
  k.block_table = block_table;
  k.seq_lens = seq_lens;
  k.win_start = win_start;
  k.window_q = static_cast<const __nv_bfloat16*>(window_q);
  char* base = static_cast<char*>(workspace);
  k.status = c->status_dev;          // library-owned, sticky until kara_status (the workspace's first 32 bytes are unused)
  k.partial = reinterpret_cast<float*>(base + w.partial_off);
  k.scores = reinterpret_cast<float*>(base + w.scores_off);
  k.idx_topk = reinterpret_cast<int32_t*>(base + w.topk_off);
  k.idx_final = reinterpret_cast<int32_t*>(base + w.final_off);
  k.n_pad = w.n_pad; k.k_pad = w.k_pad; k.keep_pad = w.keep_pad;
  k.parts = w.parts;          // strips reserved per unit; the score kernels say how many they fill
  k.part_T = k.part_nc = k.part_tpu = 0;
  k.keep_debug = (flags & KARA_KEEP_DEBUG) ? 1 : 0;
  k.free_list = c->free_list;
  k.free_count = c->free_count;

  int launches = 0;

  // ---- a1 score ------------------------------------------------------------------------------
  // One score backend: the tcgen05 / TMA kernel.  A call it cannot take is an error, not a quiet detour through the
  // CUDA-core kernel — that one runs only when the caller asks for it by name (KARA_SCORE_SIMT, a cross-check).
  if (!(flags & KARA_SCORE_SIMT) && !score_tc_supported(c->tc, k))
    return fail(KARA_EUNSUPPORTED, "the tcgen05 score kernel cannot take this call (%s); KARA_SCORE_SIMT runs the CUDA-core "
                "cross-check kernel instead, on purpose", score_tc_unsupported_reason(c->tc, k));
  const bool use_tc = !(flags & KARA_SCORE_SIMT);
  if (c->timing) {
    if (!c->ev0) { KARA_CUDA(cudaEventCreate(&c->ev0)); KARA_CUDA(cudaEventCreate(&c->ev1)); }
    KARA_CUDA(cudaEventRecord(c->ev0, st));
  }
  if (use_tc) {
    int nl = 0;
    rc = score_tc_launch(&c->tc, k, st, &nl);    // sets k.part_T / part_nc / part_tpu
    if (rc != KARA_OK) return fail(rc, "score_tc_launch: %s", score_tc_error());
    c->last_score_path = 2;
    c->last_score_reason = "";
    launches += nl;
  } else {
    const int rows = (W - k.q_row_begin) * k.G;
    const int want = (rows + 127) / 128;
    k.parts = want < w.parts ? want : w.parts;   // row parts of the SIMT kernel, all of them filled
    if (k.parts > 16) k.parts = 16;
    KARA_CUDA(launch_score_simt(k, st));
    ++launches;
    c->last_score_path = 1;
    c->last_score_reason = "KARA_SCORE_SIMT was set";
  }
  if (c->timing) { KARA_CUDA(cudaEventRecord(c->ev1, st)); c->ev_recorded = true; }

  // ---- a2-a4 select + Token2Chunk + compaction ---------------------------------------------------
  KARA_CUDA(launch_select_compact(k, st));
  ++launches;
  if (n_windows > 1) {      // prefill: the rows of all windows of a (layer, sequence, head) are moved by one CTA, in window order
    KARA_CUDA(launch_compact_windows(k, st));
    ++launches;
  }

  // ---- a5 metadata ---------------------------------------------------------------------------------
  if (flags & KARA_COMMIT) {
    KARA_CUDA(launch_metadata(k, st));
    ++launches;
  }
  c->last = k;
  c->have_last = true;
  c->last_launches = launches;
  return KARA_OK;
}

int kara_compress_window_host(kara_cache* c, int layer_begin, int layer_end, int n_seqs, int32_t* block_table,
                              int max_blocks, int32_t* seq_lens, const int32_t* win_start, const void* window_q,
                              int n_q_heads, int W, int U, double ratio, int alpha, int gamma, unsigned flags,
                              int32_t* free_count_out, void* stream) {
  int keep = 0;
  int rc = check_geometry(c, layer_begin, layer_end, n_seqs, n_q_heads, W, U, ratio, alpha, gamma, &keep);
  if (rc != KARA_OK) return rc;
  if (!block_table || !seq_lens || !window_q || max_blocks <= 0)
    return fail(KARA_EINVAL, "null host pointer or max_blocks=%d", max_blocks);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const int nL = layer_end - layer_begin;
  const size_t q_bytes = (size_t)nL * n_seqs * W * n_q_heads * c->g.d * 2;
  const size_t bt_bytes = sizeof(int32_t) * (size_t)n_seqs * max_blocks;
  const size_t sl_bytes = sizeof(int32_t) * (size_t)n_seqs;
  const size_t work_bytes = kara_workspace_bytes(c, nL, n_seqs, n_q_heads, W, U, ratio, alpha);
  auto grow = [&](void** p, size_t* have, size_t need) -> cudaError_t {
    if (*have >= need) return cudaSuccess;
    if (*p) cudaFree(*p);
    *p = nullptr; *have = 0;
    cudaError_t e = cudaMalloc(p, need);
    if (e == cudaSuccess) *have = need;
    return e;
  };
  KARA_CUDA(grow(&c->d_q, &c->d_q_bytes, q_bytes));
  KARA_CUDA(grow(reinterpret_cast<void**>(&c->d_bt), &c->d_bt_bytes, bt_bytes));
  if (c->d_sl_bytes < sl_bytes) {
    if (c->d_sl) cudaFree(c->d_sl);
    if (c->d_ws) cudaFree(c->d_ws);
    c->d_sl = c->d_ws = nullptr; c->d_sl_bytes = 0;
    KARA_CUDA(cudaMalloc(reinterpret_cast<void**>(&c->d_sl), sl_bytes));
    KARA_CUDA(cudaMalloc(reinterpret_cast<void**>(&c->d_ws), sl_bytes));
    c->d_sl_bytes = sl_bytes;
  }
  KARA_CUDA(grow(&c->d_work, &c->d_work_bytes, work_bytes));

  KARA_CUDA(cudaMemcpyAsync(c->d_q, window_q, q_bytes, cudaMemcpyHostToDevice, st));
  KARA_CUDA(cudaMemcpyAsync(c->d_bt, block_table, bt_bytes, cudaMemcpyHostToDevice, st));
  KARA_CUDA(cudaMemcpyAsync(c->d_sl, seq_lens, sl_bytes, cudaMemcpyHostToDevice, st));
  if (win_start) KARA_CUDA(cudaMemcpyAsync(c->d_ws, win_start, sl_bytes, cudaMemcpyHostToDevice, st));
  rc = kara_compress_window(c, layer_begin, layer_end, n_seqs, c->d_bt, max_blocks, c->d_sl,
                            win_start ? c->d_ws : nullptr, c->d_q, n_q_heads, W, U, ratio, alpha, gamma, flags,
                            c->d_work, c->d_work_bytes, stream);
  if (rc != KARA_OK) return rc;
  KARA_CUDA(cudaMemcpyAsync(block_table, c->d_bt, bt_bytes, cudaMemcpyDeviceToHost, st));
  KARA_CUDA(cudaMemcpyAsync(seq_lens, c->d_sl, sl_bytes, cudaMemcpyDeviceToHost, st));
  if (free_count_out)
    KARA_CUDA(cudaMemcpyAsync(free_count_out, c->free_count, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  KARA_CUDA(cudaStreamSynchronize(st));
  return KARA_OK;
}

int kara_gather_debug(kara_cache* c, int what, int layer, int seq, int kv_head, const int32_t* block_table,
                      const int32_t* seq_lens, int max_blocks, void* out, int64_t out_capacity_bytes,
                      int64_t* out_count) {
  if (!c || !out || !out_count) return fail(KARA_EINVAL, "null argument");
  *out_count = 0;
  if (!c->attached) return fail(KARA_EINVAL, "no pool attached");
  KARA_CUDA(cudaDeviceSynchronize());
  auto copy_out = [&](const void* dev, int64_t elems, int64_t elem_bytes) -> int {
    if (elems * elem_bytes > out_capacity_bytes)
      return fail(KARA_ENOMEM, "out buffer %lld bytes < %lld needed", (long long)out_capacity_bytes,
                  (long long)(elems * elem_bytes));
    if (elems > 0) KARA_CUDA(cudaMemcpy(out, dev, (size_t)(elems * elem_bytes), cudaMemcpyDeviceToHost));
    *out_count = elems;
    return KARA_OK;
  };
  switch (what) {
    case KARA_DBG_K_LOGICAL:
    case KARA_DBG_V_LOGICAL: {
      if (!block_table || !seq_lens || seq < 0 || max_blocks <= 0 || layer < 0 || layer >= c->g.n_layers ||
          kv_head < 0 || kv_head >= c->g.n_kv_heads)
        return fail(KARA_EINVAL, "bad (layer, seq, kv_head) or tables");
      int32_t len = 0;
      KARA_CUDA(cudaMemcpy(&len, seq_lens + seq, sizeof len, cudaMemcpyDeviceToHost));
      if (len < 0 || ((len + c->g.bs - 1) >> c->g.bs_log2) > max_blocks)
        return fail(KARA_EINVAL, "seq_len=%d does not fit max_blocks=%d", len, max_blocks);
      const int64_t elems = (int64_t)len * c->g.d;
      if (elems * 2 > out_capacity_bytes)
        return fail(KARA_ENOMEM, "out buffer %lld bytes < %lld needed", (long long)out_capacity_bytes,
                    (long long)(elems * 2));
      if (len == 0) return KARA_OK;
      __nv_bfloat16* tmp = nullptr;
      int32_t* st_word = nullptr;
      KARA_CUDA(cudaMalloc(reinterpret_cast<void**>(&tmp), (size_t)elems * 2));
      KARA_CUDA(cudaMalloc(reinterpret_cast<void**>(&st_word), sizeof(int32_t)));
      cudaMemset(st_word, 0, sizeof(int32_t));
      const __nv_bfloat16* pool = static_cast<const __nv_bfloat16*>(what == KARA_DBG_K_LOGICAL ? c->k_pool : c->v_pool);
      cudaError_t e = launch_gather_rows(c->g, pool, layer, kv_head, block_table + (int64_t)seq * max_blocks, len,
                                         tmp, st_word, nullptr);
      int32_t bad = 0;
      if (e == cudaSuccess) e = cudaMemcpy(out, tmp, (size_t)elems * 2, cudaMemcpyDeviceToHost);
      if (e == cudaSuccess) e = cudaMemcpy(&bad, st_word, sizeof bad, cudaMemcpyDeviceToHost);
      cudaFree(tmp);
      cudaFree(st_word);
      if (e != cudaSuccess) return fail(KARA_ECUDA, "gather: %s", cudaGetErrorString(e));
      if (bad) return fail(KARA_EINVAL, "block table row holds ids outside the pool");
      *out_count = elems;
      return KARA_OK;
    }
    case KARA_DBG_SCORES:
    case KARA_DBG_IDX_TOPK:
    case KARA_DBG_IDX_FINAL: {
      if (!c->have_last || !c->last.keep_debug)
        return fail(KARA_EINVAL, "no previous kara_compress_window call with KARA_KEEP_DEBUG");
      const Call& k = c->last;
      const int li = layer - k.layer_begin;
      // after a multi-window call `seq` is sequence * n_windows + window (include/kara.h)
      if (li < 0 || li >= k.n_layers || seq < 0 || seq >= k.n_seqs * k.n_windows || kv_head < 0 || kv_head >= k.g.n_kv_heads)
        return fail(KARA_EINVAL, "unit (layer=%d, seq=%d, head=%d) not in the last call", layer, seq, kv_head);
      const int64_t unit = ((int64_t)li * k.n_seqs * k.n_windows + seq) * k.g.n_kv_heads + kv_head;
      if (what == KARA_DBG_SCORES) return copy_out(k.scores + unit * k.n_pad, k.n, 4);
      if (what == KARA_DBG_IDX_TOPK) return copy_out(k.idx_topk + unit * k.k_pad, k.k, 4);
      return copy_out(k.idx_final + unit * k.keep_pad, k.keep, 4);
    }
    case KARA_DBG_BLOCK_TABLE_ROW:
      if (!block_table || seq < 0 || max_blocks <= 0) return fail(KARA_EINVAL, "bad table arguments");
      return copy_out(block_table + (int64_t)seq * max_blocks, max_blocks, 4);
    case KARA_DBG_FREE_LIST: {
      int32_t cnt = 0;
      KARA_CUDA(cudaMemcpy(&cnt, c->free_count, sizeof cnt, cudaMemcpyDeviceToHost));
      if (cnt < 0 || cnt > c->g.num_blocks) return fail(KARA_EINVAL, "free_count=%d out of range", cnt);
      return copy_out(c->free_list, cnt, 4);
    }
    default:
      return fail(KARA_EINVAL, "unknown what=%d", what);
  }
}

int kara_policy_step(kara_cache* c, int n_seqs, int32_t* block_table, int max_blocks, int32_t* seq_lens,
                     int32_t* uncompressed, const uint8_t* active, int32_t* step_counter, int delta, int W,
                     int max_select, int32_t* sel_ids, int32_t* sel_count, int32_t* sel_block_table,
                     int32_t* sel_seq_lens, int32_t* sel_win_start, int32_t* exhausted, void* stream) {
  if (!c || !c->attached) return fail(KARA_EINVAL, "kara_policy_step: no pool attached");
  if (n_seqs <= 0 || max_blocks <= 0 || delta <= 0 || W <= 0 || max_select <= 0)
    return fail(KARA_EINVAL, "kara_policy_step: n_seqs=%d max_blocks=%d delta=%d W=%d max_select=%d", n_seqs, max_blocks,
                delta, W, max_select);
  if (!block_table || !seq_lens || !uncompressed || !step_counter || !sel_ids || !sel_count || !sel_block_table ||
      !sel_seq_lens || !sel_win_start || !exhausted)
    return fail(KARA_EINVAL, "kara_policy_step: null pointer argument");
  KARA_CUDA(launch_policy_step(n_seqs, max_blocks, c->g.bs, c->g.bs_log2, delta, W, max_select, block_table, seq_lens,
                               uncompressed, active, c->free_list, c->free_count, step_counter, sel_ids, sel_count,
                               sel_block_table, sel_seq_lens, sel_win_start, exhausted,
                               reinterpret_cast<cudaStream_t>(stream)));
  return KARA_OK;
}

int kara_policy_commit(kara_cache* c, int max_select, const int32_t* sel_ids, const int32_t* sel_count,
                       const int32_t* sel_block_table, const int32_t* sel_seq_lens, const int32_t* sel_win_start,
                       int W, int U, double ratio, int32_t* block_table, int max_blocks, int32_t* seq_lens,
                       int32_t* uncompressed, void* stream) {
  if (!c) return fail(KARA_EINVAL, "null handle");
  if (U < 0 || W <= U || max_select <= 0 || max_blocks <= 0) return fail(KARA_EINVAL, "kara_policy_commit: bad W/U/sizes");
  const int keep = budget(W - U, ratio);
  if (keep < 0) return fail(KARA_EINVAL, "ratio=%g outside (0,1]", ratio);
  if (!sel_ids || !sel_count || !sel_block_table || !sel_seq_lens || !sel_win_start || !block_table || !seq_lens ||
      !uncompressed)
    return fail(KARA_EINVAL, "kara_policy_commit: null pointer argument");
  KARA_CUDA(launch_policy_commit(max_select, max_blocks, keep, U, W, sel_ids, sel_count, sel_block_table, sel_seq_lens,
                                 sel_win_start, block_table, seq_lens, uncompressed,
                                 reinterpret_cast<cudaStream_t>(stream)));
  return KARA_OK;
}

size_t kara_window_queries_workspace_bytes(int max_position, int head_dim) {
  if (head_dim != 64 && head_dim != 128) return 0;
  return qproj_workspace_bytes(max_position, head_dim);
}

int kara_window_queries(const void* hidden, const void* wq, const int32_t* positions, int max_position, double rope_theta,
                        int n_tokens, int d_model, int n_q_heads, int head_dim, void* window_q_out, void* workspace,
                        size_t workspace_bytes, void* stream) {
  if (!hidden || !wq || !window_q_out || n_tokens < 0 || n_q_heads <= 0)
    return fail(KARA_EINVAL, "kara_window_queries: null pointer or bad sizes");
  if (head_dim != 64 && head_dim != 128) return fail(KARA_EUNSUPPORTED, "head_dim=%d: need 64 or 128", head_dim);
  if (d_model <= 0 || d_model % 64 != 0) return fail(KARA_EUNSUPPORTED, "d_model=%d: need a positive multiple of 64", d_model);
  if (((uintptr_t)hidden | (uintptr_t)wq | (uintptr_t)window_q_out) & 15u)
    return fail(KARA_EINVAL, "kara_window_queries: hidden, wq and window_q_out must be 16-byte aligned");
  if (positions && (!workspace || max_position < 0 || !(rope_theta > 1.0)))
    return fail(KARA_EINVAL, "kara_window_queries: rotary embedding needs a workspace, max_position >= 0 and theta > 1");
  const int rc = qproj_launch(hidden, wq, positions, max_position, rope_theta, n_tokens, d_model, n_q_heads, head_dim,
                              window_q_out, workspace, workspace_bytes, reinterpret_cast<cudaStream_t>(stream));
  if (rc != KARA_OK) return fail(rc, "kara_window_queries: %s", qproj_error());
  return KARA_OK;
}

int kara_status(kara_cache* c, int32_t* status_out) {
  if (!c || !status_out) return fail(KARA_EINVAL, "null argument");
  *status_out = 0;
  if (!c->status_dev) return KARA_OK;       // no pool attached yet: nothing can have faulted
  KARA_CUDA(cudaDeviceSynchronize());
  KARA_CUDA(cudaMemcpy(status_out, c->status_dev, sizeof(int32_t), cudaMemcpyDeviceToHost));
  KARA_CUDA(cudaMemset(c->status_dev, 0, 8 * sizeof(int32_t)));
  return KARA_OK;
}

int kara_last_launch_count(const kara_cache* c) { return c ? c->last_launches : 0; }
int kara_last_score_path(const kara_cache* c) { return c ? c->last_score_path : 0; }
const char* kara_last_score_path_reason(const kara_cache* c) { return c && c->last_score_reason ? c->last_score_reason : ""; }

int kara_enable_score_timing(kara_cache* c, int enable) {
  if (!c) return fail(KARA_EINVAL, "null handle");
  c->timing = enable != 0;
  c->ev_recorded = false;
  return KARA_OK;
}

float kara_score_kernel_ms(kara_cache* c) {
  if (!c || !c->ev_recorded) return -1.f;
  if (cudaEventSynchronize(c->ev1) != cudaSuccess) return -1.f;
  float ms = -1.f;
  if (cudaEventElapsedTime(&ms, c->ev0, c->ev1) != cudaSuccess) return -1.f;
  return ms;
}

}  // extern "C"
