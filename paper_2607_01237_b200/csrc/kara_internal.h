// kara_internal.h — shared declarations of libkara's translation units (not part of the ABI).
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/kara.h"

namespace kara {

// Geometry of the paged pool (include/kara.h "Physical layout"), strides in bf16 elements.
struct Geom {
  int bs, bs_log2, n_layers, n_kv_heads, d;
  long long num_blocks;
  long long sL, sB, sH;  // layer, block, head strides; slot stride = d
};

// Parameters of one compress_window call, passed by value to every kernel.
struct Call {
  Geom g;
  const __nv_bfloat16* k_pool;
  const __nv_bfloat16* v_pool;  // written by the compaction kernel through a non-const alias
  int layer_begin, n_layers, n_seqs, max_blocks;
  int n_windows;    // NW >= 1 disjoint windows of W tokens per sequence (prefill, App. C.2; 1 = the decoding-time step)
  int n_q_heads, G, W, U, n, keep, k, P, alpha, gamma;
  int q_row_begin;  // first window token used as a query (0, or W-U with KARA_SCORE_QBUF_ONLY)
  // a 128-row query tile of the tcgen05 kernel = q_tile_toks window tokens x (1 << q_hpt_log2) query heads of the group
  // (128 x 1 normally; with KARA_SCORE_QBUF_ONLY the few buffer tokens of several heads share a tile)
  int q_tile_toks, q_hpt_log2;
  int32_t* block_table;
  int32_t* seq_lens;
  const int32_t* win_start;
  const __nv_bfloat16* window_q;
  // workspace pieces
  int32_t* status;   // [8]
  float* partial;    // [units][parts][n_pad]  (parts = strips reserved per unit)
  float* scores;     // [units][n_pad]
  int32_t* idx_topk; // [units][k_pad]
  int32_t* idx_final;// [units][keep_pad]
  int parts, n_pad, k_pad, keep_pad;
  // Which strips of a unit hold data.  part_T == 0: all `parts` strips (SIMT kernel).  part_T > 0
  // (tcgen05 kernel): the T = units*part_tpu query tiles are split into part_nc contiguous ranges,
  // one per cluster; a unit's tiles touch clusters [tile_owner(first), tile_owner(last)] and each
  // of them writes kScoreStrips strips: strips_of_unit().
  int part_T, part_nc, part_tpu;
  int keep_debug;
  int32_t* free_list;
  int32_t* free_count;
};

struct WsLayout {
  size_t status_off, partial_off, scores_off, topk_off, final_off, total;
  int parts, n_pad, k_pad, keep_pad;
};

constexpr int kScoreStrips = 1; // strips a range writes per unit
constexpr int kMaxSms = 160;    // upper bound on clusters of one launch (B200: 148 SMs)
constexpr int kMaxN = 2048;     // largest compressible region (cfg 5: 1984)

inline int round_up(int x, int m) { return (x + m - 1) / m * m; }

// Cluster that owns global query tile `tile` when T tiles are cut into nc contiguous ranges
// [floor(c T / nc), floor((c+1) T / nc)).
__host__ __device__ inline int tile_owner(long long tile, int nc, int T) {
  return (int)(((tile + 1) * nc - 1) / T);
}
// Number of partial-score strips the score kernel wrote for `unit` (see Call::part_T).
__host__ __device__ inline int strips_of_unit(int unit, int parts, int part_T, int part_nc, int part_tpu) {
  if (part_T <= 0) return parts;
  const long long first = (long long)unit * part_tpu;
  return kScoreStrips * (tile_owner(first + part_tpu - 1, part_nc, part_T) - tile_owner(first, part_nc, part_T) + 1);
}
// Upper bound of strips_of_unit over every split of units*tpu tiles into <= kMaxSms ranges: a
// range holds >= p = floor(T/nc) tiles, so the tpu consecutive tiles of a unit meet at most
// ceil((tpu-1)/p) + 1 ranges, and never more than tpu.
inline int strips_bound(int units, int tpu) {
  long long p = ((long long)units * tpu) / kMaxSms;
  if (p < 1) p = 1;
  long long ranges = (tpu - 1 + p - 1) / p + 1;
  if (ranges > tpu) ranges = tpu;
  return (int)(kScoreStrips * ranges);
}

// unit index -> (layer-in-call, sequence, window, kv head); units are ordered ((layer, sequence), window, kv head)
__host__ __device__ inline void unit_decode(int unit, int n_seqs, int n_windows, int n_kv_heads, int& li, int& s, int& w,
                                            int& hk) {
  hk = unit % n_kv_heads;
  unit /= n_kv_heads;
  w = unit % n_windows;
  unit /= n_windows;
  s = unit % n_seqs;
  li = unit / n_seqs;
}
__host__ __device__ inline int unit_count(const Call& c) { return c.n_layers * c.n_seqs * c.n_windows * c.g.n_kv_heads; }

// Window geometry of sequence s, validated on the device: h = first token of its FIRST window, t = tail tokens behind its
// last window (window w covers [h + w W, h + (w+1) W)).  Returns false (and sets status bits) if the sequence must be skipped.
__device__ inline bool window_of(const Call& c, int s, int& h, int& t, int& len) {
  len = c.seq_lens[s];
  if (len < 0) { h = 0; t = 0; return false; }     // an absent row of a kara_policy_step sub-batch: skipped silently
  h = c.win_start ? c.win_start[s] : len - c.n_windows * c.W;
  t = len - h - c.n_windows * c.W;
  int bad = 0;
  if (h < 0 || t < 0) bad |= KARA_ST_SHORT_SEQ;
  if (((len + c.g.bs - 1) >> c.g.bs_log2) > c.max_blocks) bad |= KARA_ST_TABLE_OVERFLOW;
  if (bad) { atomicOr(c.status, bad); return false; }
  return true;
}

// True if every block-table entry the window of sequence s touches — tokens [h, len), i.e. the rows the
// compaction reads or writes and the trailing entries a5 may free — is a block id inside the pool.
// Called by ALL threads of a CTA (contains __syncthreads); sets the status bit on failure.  Depends on the
// tables only, so every kernel of every call of a step takes the same decision for a sequence.
__device__ inline bool window_blocks_ok(const Call& c, int s, int h, int len) {
  const int b0 = h >> c.g.bs_log2, b1 = (len + c.g.bs - 1) >> c.g.bs_log2;
  const int32_t* row = c.block_table + (long long)s * c.max_blocks;
  int bad = 0;
  for (int b = b0 + (int)threadIdx.x; b < b1; b += (int)blockDim.x) {
    const int blk = row[b];
    bad |= (blk < 0 || blk >= c.g.num_blocks) ? 1 : 0;
  }
  bad = __syncthreads_or(bad);
  if (bad && threadIdx.x == 0) atomicOr(c.status, KARA_ST_BAD_BLOCK);
  return !bad;
}

// Element offset of logical token `pos` of sequence s, head hk, in layer `layer` (absolute).
// Returns -1 (and sets the status bit) if the block id is outside the pool.
__device__ inline long long row_offset(const Call& c, int layer, int s, int hk, int pos) {
  const int blk = c.block_table[(long long)s * c.max_blocks + (pos >> c.g.bs_log2)];
  if (blk < 0 || blk >= c.g.num_blocks) { atomicOr(c.status, KARA_ST_BAD_BLOCK); return -1; }
  return (long long)layer * c.g.sL + (long long)blk * c.g.sB + (long long)hk * c.g.sH +
         (long long)(pos & (c.g.bs - 1)) * c.g.d;
}

// sets the thread-local message kara_last_error() returns and hands `code` back (kara_api.cu)
int api_fail(int code, const char* fmt, ...);

// kernel launchers (each returns the cudaError_t of its launch)
cudaError_t launch_score_simt(const Call& c, cudaStream_t st);
cudaError_t launch_select_compact(const Call& c, cudaStream_t st);
cudaError_t launch_compact_windows(const Call& c, cudaStream_t st);   // a4 of a multi-window call (n_windows > 1)
cudaError_t launch_metadata(const Call& c, cudaStream_t st);
cudaError_t launch_policy_step(int n_seqs, int max_blocks, int bs, int bs_log2, int delta, int W, int max_select,
                               int32_t* block_table, int32_t* seq_lens, int32_t* uncompressed, const uint8_t* active,
                               int32_t* free_list, int32_t* free_count, int32_t* step_counter, int32_t* sel_ids,
                               int32_t* sel_count, int32_t* sel_block_table, int32_t* sel_seq_lens, int32_t* sel_win_start,
                               int32_t* exhausted, cudaStream_t st);
cudaError_t launch_policy_commit(int max_select, int max_blocks, int keep, int U, int W, const int32_t* sel_ids,
                                 const int32_t* sel_count, const int32_t* sel_block_table, const int32_t* sel_seq_lens,
                                 const int32_t* sel_win_start, int32_t* block_table, int32_t* seq_lens,
                                 int32_t* uncompressed, cudaStream_t st);
// window-query producer (qproj.cu): returns KARA_OK / KARA_E*; qproj_error() has the message
size_t qproj_workspace_bytes(int max_position, int d);
int qproj_launch(const void* hidden, const void* wq, const int32_t* positions, int max_position, double theta, int T,
                 int Dm, int Hq, int d, void* out, void* workspace, size_t workspace_bytes, cudaStream_t st);
const char* qproj_error();
cudaError_t launch_gather_rows(const Geom& g, const __nv_bfloat16* pool, int layer, int kv_head,
                               const int32_t* bt_row, int length, __nv_bfloat16* out, int32_t* status,
                               cudaStream_t st);

}  // namespace kara
