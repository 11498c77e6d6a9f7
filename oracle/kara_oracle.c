/*
 * kara_oracle.c — see kara_oracle.h.  TEST INFRASTRUCTURE ONLY; shares nothing with the
 * CUDA path.  Plain C99, single-threaded, fp64; every function cites the passage it follows.
 */
#include "kara_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ---------------------------------------------------------------------------------------- */

double kara_oracle_bf16_to_double(uint16_t bits) {
  /* bf16 is the upper half of an IEEE-754 binary32. */
  uint32_t u = ((uint32_t)bits) << 16;
  float f;
  memcpy(&f, &u, sizeof f);
  return (double)f;
}

/* Eq. 5: ceil(r (|W| - |U|)).  Reading G5: r is a decimal such as 0.2; the
 * 1e-9 guard keeps 0.2*480 = 96.00000000000001 from rounding up to 97. */
int kara_oracle_budget(int n, double ratio) {
  if (n <= 0 || !(ratio > 0.0) || ratio > 1.0) return KARA_ORACLE_EINVAL;
  return (int)ceil(ratio * (double)n - 1e-9);
}

/* ---------------------------------------------------------------------------------------- */
/* Eq. 4.  Queries i in [i_begin, W) x G heads, keys j in [0, n).         */

static int scores_impl(const uint16_t* q, long q_tok_stride, long q_head_stride,
                       const uint16_t* k, long k_row_stride,
                       int i_begin, int W, int G, int n, int d, double* A64, float* A32) {
  if (!q || !k || W <= 0 || G <= 0 || n <= 0 || d <= 0 || i_begin < 0 || i_begin >= W)
    return KARA_ORACLE_EINVAL;
  double* kd = (double*)malloc(sizeof(double) * (size_t)n * (size_t)d);
  double* s = (double*)malloc(sizeof(double) * (size_t)n);
  double* A = (double*)calloc((size_t)n, sizeof(double));
  double* qd = (double*)malloc(sizeof(double) * (size_t)d);
  if (!kd || !s || !A || !qd) { free(kd); free(s); free(A); free(qd); return KARA_ORACLE_EINVAL; }

  for (int j = 0; j < n; ++j)
    for (int c = 0; c < d; ++c)
      kd[(size_t)j * d + c] = kara_oracle_bf16_to_double(k[(long)j * k_row_stride + c]);

  const double inv_sqrt_d = 1.0 / sqrt((double)d);
  for (int i = i_begin; i < W; ++i) {
    for (int g = 0; g < G; ++g) {
      const uint16_t* qrow = q + (long)i * q_tok_stride + (long)g * q_head_stride;
      for (int c = 0; c < d; ++c) qd[c] = kara_oracle_bf16_to_double(qrow[c]);
      /* O1: logits of this query against every compressible key (no mask: bidirectional). */
      double m = -INFINITY;
      for (int j = 0; j < n; ++j) {
        double acc = 0.0;
        const double* kr = kd + (size_t)j * d;
        for (int c = 0; c < d; ++c) acc += qd[c] * kr[c];
        s[j] = acc * inv_sqrt_d;
        if (s[j] > m) m = s[j];
      }
      /* O2: softmax over the key dimension. */
      double l = 0.0;
      for (int j = 0; j < n; ++j) { s[j] = exp(s[j] - m); l += s[j]; }
      /* O3: colsum — accumulate this query's probabilities onto the keys. */
      for (int j = 0; j < n; ++j) A[j] += s[j] / l;
    }
  }
  for (int j = 0; j < n; ++j) {
    if (A64) A64[j] = A[j];
    if (A32) A32[j] = (float)A[j];
  }
  free(kd); free(s); free(A); free(qd);
  return KARA_ORACLE_OK;
}

int kara_oracle_scores(const uint16_t* q, long q_tok_stride, long q_head_stride,
                       const uint16_t* k, long k_row_stride,
                       int W, int G, int n, int d, double* A64, float* A32) {
  return scores_impl(q, q_tok_stride, q_head_stride, k, k_row_stride, 0, W, G, n, d, A64, A32);
}

int kara_oracle_scores_buffer_queries(const uint16_t* q, long q_tok_stride, long q_head_stride,
                                      const uint16_t* k, long k_row_stride,
                                      int W, int U, int G, int n, int d, double* A64, float* A32) {
  if (U <= 0 || U > W) return KARA_ORACLE_EINVAL;
  return scores_impl(q, q_tok_stride, q_head_stride, k, k_row_stride, W - U, W, G, n, d, A64, A32);
}

/* ---------------------------------------------------------------------------------------- */
/* Eq. 5-8 + App. C.3.                                                                         */

typedef struct { float v; int32_t i; } scored;

/* total order: value descending, then index ascending (reading G4) */
static int cmp_scored(const void* pa, const void* pb) {
  const scored* a = (const scored*)pa;
  const scored* b = (const scored*)pb;
  if (a->v > b->v) return -1;
  if (a->v < b->v) return 1;
  return (a->i > b->i) - (a->i < b->i);
}
static int cmp_int32(const void* pa, const void* pb) {
  int32_t a = *(const int32_t*)pa, b = *(const int32_t*)pb;
  return (a > b) - (a < b);
}

int kara_oracle_select(const float* A32, int n, int keep, int alpha, int gamma,
                       int32_t* I_out, int32_t* chunks_out, int32_t* F_out,
                       int32_t* n_chunk_added_out) {
  if (!A32 || n <= 0 || alpha < 0) return KARA_ORACLE_EINVAL;
  const int k = keep - alpha;
  if (gamma < 3 || k < 1 || keep > n) return KARA_ORACLE_EBUDGET; /* PAPER.md:L140 gamma >= 3 */
  const int P = alpha / (gamma - 2);                              /* Eq. 7 floor(alpha/(gamma-2)) */

  scored* order = (scored*)malloc(sizeof(scored) * (size_t)n);
  int32_t* I = (int32_t*)malloc(sizeof(int32_t) * (size_t)k);
  unsigned char* kept = (unsigned char*)calloc((size_t)n, 1);
  scored* R = (scored*)malloc(sizeof(scored) * (size_t)(k > 1 ? k - 1 : 1));
  if (!order || !I || !kept || !R) { free(order); free(I); free(kept); free(R); return KARA_ORACLE_EINVAL; }

  /* O5 (Eq. 5): the k best-scoring positions, then sorted ascending. */
  for (int j = 0; j < n; ++j) { order[j].v = A32[j]; order[j].i = j; }
  qsort(order, (size_t)n, sizeof(scored), cmp_scored);
  for (int t = 0; t < k; ++t) I[t] = order[t].i;
  qsort(I, (size_t)k, sizeof(int32_t), cmp_int32);
  for (int t = 0; t < k; ++t) kept[I[t]] = 1;

  /* O6 (Eq. 6) + the constraint of Eq. 7: candidate chunk t has endpoints I[t], I[t+1]. */
  int n_elig = 0;
  for (int t = 0; t + 1 < k; ++t) {
    const int a = I[t], b = I[t + 1];
    const int gap = b - a - 1;
    if (b - a < gamma && gap >= 1) {
      volatile float sum = A32[a] + A32[b];          /* fl32 add  (reading G14) */
      volatile float r = sum * (float)gap;           /* fl32 mul, no contraction */
      R[n_elig].v = r;
      R[n_elig].i = t;
      ++n_elig;
    }
  }
  /* O7 (Eq. 7): filter first, then the top-P chunks by R. */
  qsort(R, (size_t)n_elig, sizeof(scored), cmp_scored);
  const int n_pick = n_elig < P ? n_elig : P;
  /* O8 (Eq. 8): union the interiors of the chosen chunks with I. */
  int added = 0;
  for (int c = 0; c < n_pick; ++c) {
    const int t = R[c].i;
    for (int j = I[t] + 1; j < I[t + 1]; ++j) { kept[j] = 1; ++added; }
  }
  if (chunks_out)
    for (int c = 0; c < P; ++c) chunks_out[c] = c < n_pick ? R[c].i : -1;

  /* O9 (App. C.3): fill the rest of the chunk budget with the best-scoring
   * unselected positions of the compressible region. */
  int fill = keep - (k + added);
  for (int r = 0; r < n && fill > 0; ++r) {
    const int j = order[r].i;
    if (!kept[j]) { kept[j] = 1; --fill; }
  }

  if (I_out) memcpy(I_out, I, sizeof(int32_t) * (size_t)k);
  if (F_out) {
    int c = 0;
    for (int j = 0; j < n; ++j) if (kept[j]) F_out[c++] = j;
    if (c != keep) { free(order); free(I); free(kept); free(R); return KARA_ORACLE_EINVAL; }
  }
  if (n_chunk_added_out) *n_chunk_added_out = added;
  free(order); free(I); free(kept); free(R);
  return KARA_ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------- */
/* Eq. 9 on logical rows; buffer + tail rows follow (reading G11).             */

int kara_oracle_compact_rows(const uint16_t* old_rows, int h, int W, int U, int t, int d,
                             const int32_t* F, int keep, uint16_t* new_rows) {
  if (!old_rows || !new_rows || !F || h < 0 || U < 0 || W <= U || t < 0 || d <= 0 || keep < 0)
    return KARA_ORACLE_EINVAL;
  const int n = W - U;
  const size_t rb = sizeof(uint16_t) * (size_t)d;
  memcpy(new_rows, old_rows, rb * (size_t)h);                        /* history untouched */
  for (int c = 0; c < keep; ++c) {
    if (F[c] < 0 || F[c] >= n) return KARA_ORACLE_EINVAL;
    memcpy(new_rows + (size_t)(h + c) * d, old_rows + (size_t)(h + F[c]) * d, rb);
  }
  memcpy(new_rows + (size_t)(h + keep) * d, old_rows + (size_t)(h + n) * d, rb * (size_t)(U + t));
  return KARA_ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------- */
/* Alg. 1 l.12 UpdateMetadata + block release.                     */

static int ceil_div(int a, int b) { return (a + b - 1) / b; }

int kara_oracle_metadata(int n_seqs, int max_blocks, int block_size,
                         int32_t* block_table, int32_t* seq_lens, const int32_t* win_start,
                         int W, int U, int keep, int32_t* free_list, int32_t* free_count) {
  if (!block_table || !seq_lens || !free_list || !free_count || block_size <= 0)
    return KARA_ORACLE_EINVAL;
  for (int s = 0; s < n_seqs; ++s) {
    const int len = seq_lens[s];
    const int h = win_start ? win_start[s] : len - W;
    const int t = len - h - W;
    if (h < 0 || t < 0) return KARA_ORACLE_EINVAL;
    const int new_len = h + keep + U + t;
    const int old_nb = ceil_div(len, block_size);
    const int new_nb = ceil_div(new_len, block_size);
    if (old_nb > max_blocks) return KARA_ORACLE_EINVAL;
    for (int b = new_nb; b < old_nb; ++b) {
      free_list[(*free_count)++] = block_table[(long)s * max_blocks + b];
      block_table[(long)s * max_blocks + b] = -1;
    }
    seq_lens[s] = new_len;
  }
  return KARA_ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------- */
/* Whole path over a paged pool image.                                                         */

static uint16_t* row_ptr(const kara_oracle_layout* lay, uint16_t* pool, int layer,
                         const int32_t* bt_row, int pos, int head) {
  const int blk = bt_row[pos / lay->block_size];
  const int slot = pos % lay->block_size;
  return pool + (long)layer * lay->sL + (long)blk * lay->sB + (long)head * lay->sH +
         (long)slot * lay->sS;
}

int kara_oracle_compress_window(const kara_oracle_layout* lay, uint16_t* k_pool, uint16_t* v_pool,
                                int layer_begin, int layer_end, int n_seqs,
                                int32_t* block_table, int max_blocks, int32_t* seq_lens,
                                const int32_t* win_start,
                                const uint16_t* window_q, int n_q_heads,
                                int W, int U, double ratio, int alpha, int gamma, int commit,
                                int32_t* free_list, int32_t* free_count,
                                const float* scores_in, float* scores_out,
                                int32_t* idx_topk_out, int32_t* idx_final_out) {
  if (!lay || !k_pool || !v_pool || !block_table || !seq_lens) return KARA_ORACLE_EINVAL;
  if (!window_q && !scores_in) return KARA_ORACLE_EINVAL;
  const int d = lay->head_dim, Hkv = lay->n_kv_heads, bs = lay->block_size;
  if (layer_begin < 0 || layer_end > lay->n_layers || layer_begin >= layer_end) return KARA_ORACLE_EINVAL;
  if (n_q_heads % Hkv != 0 || U < 0 || W <= U) return KARA_ORACLE_EINVAL;
  const int G = n_q_heads / Hkv;
  const int n = W - U;
  const int keep = kara_oracle_budget(n, ratio);                      /* O4 */
  if (keep < 0) return KARA_ORACLE_EINVAL;
  const int k = keep - alpha;
  if (gamma < 3 || k < 1 || keep > n) return KARA_ORACLE_EBUDGET;
  const int nL = layer_end - layer_begin;

  uint16_t* kwin = (uint16_t*)malloc(sizeof(uint16_t) * (size_t)n * d);
  float* A32 = (float*)malloc(sizeof(float) * (size_t)n);
  int32_t* I = (int32_t*)malloc(sizeof(int32_t) * (size_t)k);
  int32_t* F = (int32_t*)malloc(sizeof(int32_t) * (size_t)keep);
  uint16_t* tmp = NULL;
  int rc = KARA_ORACLE_OK;
  if (!kwin || !A32 || !I || !F) { rc = KARA_ORACLE_EINVAL; goto done; }

  for (int li = 0; li < nL && rc == KARA_ORACLE_OK; ++li) {
    const int layer = layer_begin + li;
    for (int s = 0; s < n_seqs && rc == KARA_ORACLE_OK; ++s) {
      const int len = seq_lens[s];
      const int h = win_start ? win_start[s] : len - W;
      const int t = len - h - W;
      if (h < 0 || t < 0 || ceil_div(len, bs) > max_blocks) { rc = KARA_ORACLE_EINVAL; break; }
      const int32_t* bt_row = block_table + (long)s * max_blocks;
      const int moved = keep + U + t;     /* rows rewritten behind the history */
      tmp = (uint16_t*)realloc(tmp, sizeof(uint16_t) * (size_t)(moved > 0 ? moved : 1) * d);
      if (!tmp) { rc = KARA_ORACLE_EINVAL; break; }
      for (int hk = 0; hk < Hkv; ++hk) {
        const long unit = ((long)li * n_seqs + s) * Hkv + hk;
        if (scores_in) {
          memcpy(A32, scores_in + unit * n, sizeof(float) * (size_t)n);
        } else {
          /* K_{W\U}: logical rows [h, h+n) of this head, read through the block table. */
          for (int j = 0; j < n; ++j)
            memcpy(kwin + (size_t)j * d, row_ptr(lay, k_pool, layer, bt_row, h + j, hk),
                   sizeof(uint16_t) * (size_t)d);
          const uint16_t* q = window_q + (((long)li * n_seqs + s) * W) * n_q_heads * d +
                              (long)hk * G * d;
          rc = kara_oracle_scores(q, (long)n_q_heads * d, d, kwin, d, W, G, n, d, NULL, A32);
          if (rc) break;
        }
        if (scores_out) memcpy(scores_out + unit * n, A32, sizeof(float) * (size_t)n);
        rc = kara_oracle_select(A32, n, keep, alpha, gamma, I, NULL, F, NULL);
        if (rc) break;
        if (idx_topk_out) memcpy(idx_topk_out + unit * k, I, sizeof(int32_t) * (size_t)k);
        if (idx_final_out) memcpy(idx_final_out + unit * keep, F, sizeof(int32_t) * (size_t)keep);
        /* O10 (Eq. 9 + MemoryCompaction): gather into tmp, then lay the rows down densely at
         * logical positions [h, h+keep+U+t) through the same block table. */
        for (int which = 0; which < 2; ++which) {
          uint16_t* pool = which == 0 ? k_pool : v_pool;
          for (int c = 0; c < keep; ++c)
            memcpy(tmp + (size_t)c * d, row_ptr(lay, pool, layer, bt_row, h + F[c], hk),
                   sizeof(uint16_t) * (size_t)d);
          for (int c = 0; c < U + t; ++c)
            memcpy(tmp + (size_t)(keep + c) * d, row_ptr(lay, pool, layer, bt_row, h + n + c, hk),
                   sizeof(uint16_t) * (size_t)d);
          for (int c = 0; c < moved; ++c)
            memcpy(row_ptr(lay, pool, layer, bt_row, h + c, hk), tmp + (size_t)c * d,
                   sizeof(uint16_t) * (size_t)d);
        }
      }
    }
  }
  if (rc == KARA_ORACLE_OK && commit)
    rc = kara_oracle_metadata(n_seqs, max_blocks, bs, block_table, seq_lens, win_start, W, U, keep,
                              free_list, free_count);
done:
  free(kwin); free(A32); free(I); free(F); free(tmp);
  return rc;
}

/* ---------------------------------------------------------------------------------------- */
/* App. C.2 prefill: "partition the prompt into multiple windows of length |W|
 * and perform window-wise compression on the KV pairs corresponding to positions inside each
 * window in parallel".  Reading G17: the NW windows of a sequence are the disjoint
 * ranges [h + w W, h + (w+1) W), each scored with its own W queries against its own n keys and
 * selected on its own (O1-O9 unchanged); the retained rows and the buffer of window w are laid
 * down behind those of window w-1, the tail behind the last window:
 *   new[h + w (keep+U) + c]        = old[h + w W + F_w[c]]       c < keep
 *   new[h + w (keep+U) + keep + c] = old[h + w W + n + c]        c < U
 *   new[h + NW (keep+U) + c]       = old[h + NW W + c]           c < t
 * Unit order of every dump: ((layer, sequence), window, KV head). */
int kara_oracle_compress_windows(const kara_oracle_layout* lay, uint16_t* k_pool, uint16_t* v_pool,
                                 int layer_begin, int layer_end, int n_seqs,
                                 int32_t* block_table, int max_blocks, int32_t* seq_lens,
                                 const int32_t* win_start, int n_windows,
                                 const uint16_t* window_q, int n_q_heads,
                                 int W, int U, double ratio, int alpha, int gamma, int commit,
                                 int32_t* free_list, int32_t* free_count,
                                 const float* scores_in, float* scores_out,
                                 int32_t* idx_topk_out, int32_t* idx_final_out) {
  if (!lay || !k_pool || !v_pool || !block_table || !seq_lens) return KARA_ORACLE_EINVAL;
  if (!window_q && !scores_in) return KARA_ORACLE_EINVAL;
  const int d = lay->head_dim, Hkv = lay->n_kv_heads, bs = lay->block_size;
  if (layer_begin < 0 || layer_end > lay->n_layers || layer_begin >= layer_end) return KARA_ORACLE_EINVAL;
  if (n_q_heads % Hkv != 0 || U < 0 || W <= U || n_windows < 1) return KARA_ORACLE_EINVAL;
  const int G = n_q_heads / Hkv, NW = n_windows;
  const int n = W - U;
  const int keep = kara_oracle_budget(n, ratio);
  if (keep < 0) return KARA_ORACLE_EINVAL;
  const int k = keep - alpha;
  if (gamma < 3 || k < 1 || keep > n) return KARA_ORACLE_EBUDGET;
  const int nL = layer_end - layer_begin;
  const int per = keep + U;                       /* rows one window leaves behind */

  uint16_t* kwin = (uint16_t*)malloc(sizeof(uint16_t) * (size_t)n * d);
  float* A32 = (float*)malloc(sizeof(float) * (size_t)n);
  int32_t* I = (int32_t*)malloc(sizeof(int32_t) * (size_t)k);
  int32_t* F = (int32_t*)malloc(sizeof(int32_t) * (size_t)keep * NW);
  uint16_t* tmp = NULL;
  int rc = KARA_ORACLE_OK;
  if (!kwin || !A32 || !I || !F) { rc = KARA_ORACLE_EINVAL; goto done; }

  for (int li = 0; li < nL && rc == KARA_ORACLE_OK; ++li) {
    const int layer = layer_begin + li;
    for (int s = 0; s < n_seqs && rc == KARA_ORACLE_OK; ++s) {
      const int len = seq_lens[s];
      const int h = win_start ? win_start[s] : len - NW * W;
      const int t = len - h - NW * W;
      if (h < 0 || t < 0 || ceil_div(len, bs) > max_blocks) { rc = KARA_ORACLE_EINVAL; break; }
      const int32_t* bt_row = block_table + (long)s * max_blocks;
      const int moved = NW * per + t;
      tmp = (uint16_t*)realloc(tmp, sizeof(uint16_t) * (size_t)(moved > 0 ? moved : 1) * d);
      if (!tmp) { rc = KARA_ORACLE_EINVAL; break; }
      for (int hk = 0; hk < Hkv && rc == KARA_ORACLE_OK; ++hk) {
        for (int w = 0; w < NW; ++w) {            /* O1-O9 per window, independently */
          const long unit = (((long)li * n_seqs + s) * NW + w) * Hkv + hk;
          const int hw = h + w * W;
          if (scores_in) {
            memcpy(A32, scores_in + unit * n, sizeof(float) * (size_t)n);
          } else {
            for (int j = 0; j < n; ++j)
              memcpy(kwin + (size_t)j * d, row_ptr(lay, k_pool, layer, bt_row, hw + j, hk),
                     sizeof(uint16_t) * (size_t)d);
            const uint16_t* q = window_q + ((((long)li * n_seqs + s) * NW + w) * W) * n_q_heads * d +
                                (long)hk * G * d;
            rc = kara_oracle_scores(q, (long)n_q_heads * d, d, kwin, d, W, G, n, d, NULL, A32);
            if (rc) break;
          }
          if (scores_out) memcpy(scores_out + unit * n, A32, sizeof(float) * (size_t)n);
          rc = kara_oracle_select(A32, n, keep, alpha, gamma, I, NULL, F + (size_t)w * keep, NULL);
          if (rc) break;
          if (idx_topk_out) memcpy(idx_topk_out + unit * k, I, sizeof(int32_t) * (size_t)k);
          if (idx_final_out)
            memcpy(idx_final_out + unit * keep, F + (size_t)w * keep, sizeof(int32_t) * (size_t)keep);
        }
        if (rc) break;
        /* O10 over all windows of this (layer, head): gather, then lay down densely */
        for (int which = 0; which < 2; ++which) {
          uint16_t* pool = which == 0 ? k_pool : v_pool;
          for (int w = 0; w < NW; ++w) {
            for (int c = 0; c < keep; ++c)
              memcpy(tmp + (size_t)(w * per + c) * d,
                     row_ptr(lay, pool, layer, bt_row, h + w * W + F[(size_t)w * keep + c], hk),
                     sizeof(uint16_t) * (size_t)d);
            for (int c = 0; c < U; ++c)
              memcpy(tmp + (size_t)(w * per + keep + c) * d,
                     row_ptr(lay, pool, layer, bt_row, h + w * W + n + c, hk), sizeof(uint16_t) * (size_t)d);
          }
          for (int c = 0; c < t; ++c)
            memcpy(tmp + (size_t)(NW * per + c) * d, row_ptr(lay, pool, layer, bt_row, h + NW * W + c, hk),
                   sizeof(uint16_t) * (size_t)d);
          for (int c = 0; c < moved; ++c)
            memcpy(row_ptr(lay, pool, layer, bt_row, h + c, hk), tmp + (size_t)c * d,
                   sizeof(uint16_t) * (size_t)d);
        }
      }
    }
  }
  if (rc == KARA_ORACLE_OK && commit) {
    /* O11 with new_len = h + NW (keep+U) + t: trailing table entries freed in table order, batch order */
    for (int s = 0; s < n_seqs; ++s) {
      const int len = seq_lens[s];
      const int h = win_start ? win_start[s] : len - NW * W;
      const int t = len - h - NW * W;
      const int new_len = h + NW * per + t;
      const int old_nb = ceil_div(len, bs), new_nb = ceil_div(new_len, bs);
      for (int b = new_nb; b < old_nb; ++b) {
        free_list[(*free_count)++] = block_table[(long)s * max_blocks + b];
        block_table[(long)s * max_blocks + b] = -1;
      }
      seq_lens[s] = new_len;
    }
  }
done:
  free(kwin); free(A32); free(I); free(F); free(tmp);
  return rc;
}

/* ---------------------------------------------------------------------------------------- */
/* Alg. 1 (reading G12) + App. C.4 (L352-354): one decoding step of the periodic policy. */
int kara_oracle_policy_step(int n_seqs, int max_blocks, int block_size, int32_t* block_table, int32_t* seq_lens,
                            int32_t* uncompressed, const uint8_t* active, int32_t* free_list, int32_t* free_count,
                            int32_t* step_counter, int delta, int W, int max_select,
                            int32_t* sel_ids, int32_t* sel_count, int32_t* sel_block_table, int32_t* sel_seq_lens,
                            int32_t* sel_win_start, int32_t* exhausted) {
  if (n_seqs < 0 || max_blocks <= 0 || block_size <= 0 || delta <= 0 || W <= 0 || max_select < 0)
    return KARA_ORACLE_EINVAL;
  /* l.2: one generated token per active sequence */
  for (int s = 0; s < n_seqs; ++s) {
    if (active && !active[s]) continue;
    const int len = seq_lens[s];
    if (len % block_size == 0) {                       /* the token opens a new block */
      const int b = len / block_size;
      if (b >= max_blocks || *free_count <= 0) { if (exhausted) ++*exhausted; continue; }
      block_table[(long)s * max_blocks + b] = free_list[--*free_count];      /* pop from the top of the stack */
    }
    seq_lens[s] = len + 1;
    uncompressed[s] += 1;
  }
  /* l.3 */
  *step_counter += 1;
  const int g = *step_counter;
  /* l.4-5 */
  int cnt = 0;
  if (g > W && g % delta == 0) {
    for (int s = 0; s < n_seqs && cnt < max_select; ++s) {
      if (active && !active[s]) continue;
      const int len = seq_lens[s];
      const int t = len % block_size;                  /* the last (possibly partial) block is excluded */
      if (uncompressed[s] - t < W) continue;
      sel_ids[cnt] = s;
      sel_win_start[cnt] = len - t - W;
      sel_seq_lens[cnt] = len;
      memcpy(sel_block_table + (long)cnt * max_blocks, block_table + (long)s * max_blocks,
             sizeof(int32_t) * (size_t)max_blocks);
      ++cnt;
    }
  }
  for (int x = cnt; x < max_select; ++x) {
    sel_ids[x] = -1;
    sel_seq_lens[x] = -1;
    sel_win_start[x] = 0;
    for (int b = 0; b < max_blocks; ++b) sel_block_table[(long)x * max_blocks + b] = -1;
  }
  *sel_count = cnt;
  return KARA_ORACLE_OK;
}

/* Alg. 1 l.12 UpdateMetadata(e) for the running queue + the uncompressed-tail counter of App. C.4 (L354). */
int kara_oracle_policy_commit(int max_blocks, const int32_t* sel_ids, int sel_count, const int32_t* sel_block_table,
                              const int32_t* sel_seq_lens, const int32_t* sel_win_start, int keep, int U,
                              int32_t* block_table, int32_t* seq_lens, int32_t* uncompressed) {
  for (int x = 0; x < sel_count; ++x) {
    const int s = sel_ids[x];
    if (s < 0) return KARA_ORACLE_EINVAL;
    memcpy(block_table + (long)s * max_blocks, sel_block_table + (long)x * max_blocks,
           sizeof(int32_t) * (size_t)max_blocks);
    seq_lens[s] = sel_seq_lens[x];
    const int t = sel_seq_lens[x] - (sel_win_start[x] + keep + U);
    uncompressed[s] = U + t;
  }
  return KARA_ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------- */
/* App. C.2 query projection + rotary embedding (reading G19). */
static uint16_t double_to_bf16_rne(double x) {
  float f = (float)x;                       /* double -> float is exact enough: a bf16 keeps 8 of the float's 24 bits */
  uint32_t u;
  memcpy(&u, &f, sizeof u);
  if ((u & 0x7f800000u) == 0x7f800000u) return (uint16_t)(u >> 16);       /* inf / nan */
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

int kara_oracle_window_queries(const uint16_t* hidden, const uint16_t* wq, const int32_t* positions, double rope_theta,
                               int T, int d_model, int n_q_heads, int d, uint16_t* out) {
  if (!hidden || !wq || !out || T < 0 || d_model <= 0 || n_q_heads <= 0 || d <= 0 || (d & 1)) return KARA_ORACLE_EINVAL;
  double* q = (double*)malloc(sizeof(double) * (size_t)d);
  if (!q) return KARA_ORACLE_EINVAL;
  for (int t = 0; t < T; ++t) {
    for (int h = 0; h < n_q_heads; ++h) {
      for (int c = 0; c < d; ++c) {
        const uint16_t* wrow = wq + ((long)h * d + c) * d_model;
        double acc = 0.0;
        for (int k = 0; k < d_model; ++k)
          acc += kara_oracle_bf16_to_double(hidden[(long)t * d_model + k]) * kara_oracle_bf16_to_double(wrow[k]);
        q[c] = acc;
      }
      uint16_t* o = out + ((long)t * n_q_heads + h) * d;
      if (!positions) {
        for (int c = 0; c < d; ++c) o[c] = double_to_bf16_rne(q[c]);
      } else {
        for (int c = 0; c < d / 2; ++c) {
          const double a = (double)positions[t] * pow(rope_theta, -2.0 * (double)c / (double)d);
          const double cs = cos(a), sn = sin(a);
          o[c] = double_to_bf16_rne(q[c] * cs - q[c + d / 2] * sn);
          o[c + d / 2] = double_to_bf16_rne(q[c + d / 2] * cs + q[c] * sn);
        }
      }
    }
  }
  free(q);
  return KARA_ORACLE_OK;
}
