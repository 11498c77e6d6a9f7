/*
 * kara_oracle.h — CPU oracle for Kara's sliding-window KV-cache compression step.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this.  The product
 * (paper_2607_01237_b200/, include/kara.h) never includes, links or imports it, and this
 * file includes nothing from the product.
 *
 * Plain, single-threaded, fp64 restatement of PAPER.md (arxiv/paper_2607_01237):
 *   Eq. 4  A = colsum(softmax(Q_W K_{W\U}^T / sqrt(d)))
 *   Eq. 5  I = TopK(A, ceil(r(|W|-|U|)) - alpha)
 *   Eq. 6  R_k = (A_I[k] + A_I[k+1]) * (I[k+1] - I[k] - 1)
 *   Eq. 7  P = TopK(R, floor(alpha/(gamma-2)))  s.t. I[k+1]-I[k] < gamma
 *   Eq. 8  I^ = I u U_{k in P} { j | I[k] < j < I[k+1] }
 *   App. C.3 fill the chunk budget with best unselected discrete positions
 *   Eq. 9  (K,V)_{W\U} <- (K,V)_{W\U}[I^]
 *   Sec 4.3 / Alg. 1 l.11-12 / App. C.4 compaction + block release
 * No blocking, fusion or reordering beyond what those passages state.  Readings of the
 * places where the paper is silent (GQA sum, tie-breaks, rounding of ceil(r n), order of
 * retained rows, free-list order, prefill windows, policy order) are the ones listed in DESIGN.md "Readings" (G1..G18).
 *
 * Pins (tests/test_oracle_*.py): library float64 softmax on small cases, closed forms
 * (Q = 0, equal keys, one-hot), invariants (sum_j A_j = G*W), equivariances, integer
 * budget table, brute-force Token2Chunk on tiny n, hand-worked vectors under tests/golden/,
 * closed-form freed-block counts; the policy step against a token-level simulation (every token carries its own
 * "compressed" flag) and the paper's KvLLM numbers (B.1).  End-to-end against outputs printed by the paper:
 * PARITY UNPINNED — the paper prints no scores, indices or bytes for any input.
 *
 * Notation (window-relative, 0-based): W window length, U protected buffer at the window's
 * end, n = W-U compressible keys, G = Hq/Hkv query heads per KV head, d head_dim,
 * keep = ceil(r n), k = keep - alpha, P = floor(alpha/(gamma-2)), h = win_start (tokens in
 * front of the window, never touched), t = seq_len - (h+W) tail tokens after the window.
 */
#ifndef KARA_ORACLE_H
#define KARA_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define KARA_ORACLE_OK 0
#define KARA_ORACLE_EINVAL (-1)
#define KARA_ORACLE_EBUDGET (-2)

/* bf16 bit pattern -> double (exact widening). */
double kara_oracle_bf16_to_double(uint16_t bits);

/* O4 (Eq. 5): keep = ceil(r * n), evaluated on the decimal the caller meant:
 * (int)ceil(ratio*n - 1e-9) with ratio a double (reading G5). */
int kara_oracle_budget(int n, double ratio);

/* O1-O3 (Eq. 4): importance scores of the n compressible keys of ONE (sequence, layer,
 * KV head) unit.  q: bf16 bits; query row (i,g), i in [0,W), g in [0,G), starts at
 * q + i*q_tok_stride + g*q_head_stride (strides in elements).  k: bf16 bits, key j starts at
 * k + j*k_row_stride.  All arithmetic in double: logits s = (q.k)/sqrt(d); row softmax over
 * j (max-subtracted); A[j] = sum_i sum_g p[(i,g),j] in the fixed order i-major, g-minor;
 * A32[j] = (float)A64[j] rounded once.  Either output may be NULL. */
int kara_oracle_scores(const uint16_t* q, long q_tok_stride, long q_head_stride,
                       const uint16_t* k, long k_row_stride,
                       int W, int G, int n, int d, double* A64, float* A32);

/* Ablation "w/o Bi-Attention": same, but only the last U window tokens
 * (the buffer) act as queries: i in [W-U, W). */
int kara_oracle_scores_buffer_queries(const uint16_t* q, long q_tok_stride, long q_head_stride,
                                      const uint16_t* k, long k_row_stride,
                                      int W, int U, int G, int n, int d, double* A64, float* A32);

/* O5-O9 (Eq. 5-8 + App. C.3) from fp32 scores.  Outputs (each may be NULL):
 *   I      [keep-alpha]  candidate indices, ascending            (Eq. 5)
 *   chunks [P]           chosen chunk ordinals t (chunk t has endpoints I[t], I[t+1]),
 *                        in order of choice (R descending, t ascending); -1 padded  (Eq. 7)
 *   F      [keep]        final retained indices, ascending       (Eq. 8 + C.3 fill)
 *   n_chunk_added        number of interior positions added by Eq. 8
 * Total orders (reading G4): scores (A32 descending, index ascending); chunks (R descending,
 * ordinal ascending), R_t = fl32(fl32(A32[a]+A32[b]) * (float)(b-a-1)) (reading G14);
 * eligible iff b-a < gamma and b-a-1 >= 1 (readings G7, G8).
 * Returns KARA_ORACLE_EBUDGET unless 1 <= keep-alpha and keep <= n and gamma >= 3. */
int kara_oracle_select(const float* A32, int n, int keep, int alpha, int gamma,
                       int32_t* I, int32_t* chunks, int32_t* F, int32_t* n_chunk_added);

/* O10 (Eq. 9) on the logical rows of one (layer, KV head) of one sequence:
 * old_rows [h+W+t][d] -> new_rows [h+keep+U+t][d]:
 *   old[0:h] || old[h+F[0]], ..., old[h+F[keep-1]] || old[h+n : h+W+t]. */
int kara_oracle_compact_rows(const uint16_t* old_rows, int h, int W, int U, int t, int d,
                             const int32_t* F, int keep, uint16_t* new_rows);

/* Physical addressing of a paged pool image held in host memory, as element strides:
 * element (layer, block, kv_head, slot, c) of K (or V) is at
 *   pool[layer*sL + block*sB + kv_head*sH + slot*sS + c].
 * The caller states the strides; the oracle has no opinion on the layout. */
typedef struct {
  int block_size, n_layers, n_kv_heads, head_dim;
  long sL, sB, sH, sS;
  long num_blocks;
} kara_oracle_layout;

/* O11 (Alg. 1 l.12 "UpdateMetadata", App. C.4): per sequence s, in batch order:
 *   h = win_start[s] (NULL => seq_lens[s]-W), t = seq_lens[s]-h-W,
 *   new_len = h+keep+U+t, new_nb = ceil(new_len/bs), old_nb = ceil(seq_lens[s]/bs);
 *   block_table[s][new_nb:old_nb] appended to free_list at *free_count (table order),
 *   entries set to -1, seq_lens[s] = new_len.  (reading G16) */
int kara_oracle_metadata(int n_seqs, int max_blocks, int block_size,
                         int32_t* block_table, int32_t* seq_lens, const int32_t* win_start,
                         int W, int U, int keep, int32_t* free_list, int32_t* free_count);

/* The whole path O1-O11 over a host image of the paged pool, for layers
 * [layer_begin, layer_end) x n_seqs sequences x all KV heads.
 *   window_q   bf16 bits [layer_end-layer_begin][n_seqs][W][n_q_heads][d]
 *   scores_in  NULL, or fp32 [layers][n_seqs][n_kv_heads][n]: skip O1-O3 and run O4-O11 from
 *              these scores ("scores-injected" mode used for stage-S2 parity)
 *   scores_out / idx_topk_out [..][k] / idx_final_out [..][keep]: optional dumps, same unit order
 *   commit     nonzero => run O11 after compaction (block tables, seq_lens, free list)
 * K and V rows are moved in place inside the pool image (through block_table, rows read into a
 * temporary first, so the result is the definition of Eq. 9, not an in-place algorithm). */
int kara_oracle_compress_window(const kara_oracle_layout* lay, uint16_t* k_pool, uint16_t* v_pool,
                                int layer_begin, int layer_end, int n_seqs,
                                int32_t* block_table, int max_blocks, int32_t* seq_lens,
                                const int32_t* win_start,
                                const uint16_t* window_q, int n_q_heads,
                                int W, int U, double ratio, int alpha, int gamma, int commit,
                                int32_t* free_list, int32_t* free_count,
                                const float* scores_in, float* scores_out,
                                int32_t* idx_topk_out, int32_t* idx_final_out);

/* Prefill (App. C.2; reading G17): n_windows disjoint windows of W tokens per
 * sequence starting at win_start[s] (NULL => seq_len - n_windows*W), each compressed on its own
 * (O1-O9), retained rows + buffer of window w laid down behind those of window w-1, tail last;
 * new_len = h + n_windows*(keep+U) + t.  window_q is [layers][n_seqs][n_windows*W][n_q_heads][d];
 * dumps and scores_in are ordered ((layer, sequence), window, KV head).  n_windows = 1 is
 * kara_oracle_compress_window. */
int kara_oracle_compress_windows(const kara_oracle_layout* lay, uint16_t* k_pool, uint16_t* v_pool,
                                 int layer_begin, int layer_end, int n_seqs,
                                 int32_t* block_table, int max_blocks, int32_t* seq_lens,
                                 const int32_t* win_start, int n_windows,
                                 const uint16_t* window_q, int n_q_heads,
                                 int W, int U, double ratio, int alpha, int gamma, int commit,
                                 int32_t* free_list, int32_t* free_count,
                                 const float* scores_in, float* scores_out,
                                 int32_t* idx_topk_out, int32_t* idx_final_out);

/* Periodic compression policy (Alg. 1, reconstructed per reading G12; App. C.4; B.1, L275),
 * the bookkeeping of ONE decoding step for a batch of running sequences, in Alg. 1's order:
 *   l.2  every active sequence has generated one token: if its current length is a multiple of the block size the
 *        token opens a new block, popped from the TOP of the free-list stack (sequences in batch order; reading G18);
 *        seq_len += 1, uncompressed += 1.  A sequence that needs a block while the free list is empty is not advanced
 *        and *exhausted is incremented (the serving engine would preempt it: out of scope).
 *   l.3  g <- g + 1
 *   l.4  if g > W and g mod delta == 0:
 *   l.5    SELECT: sequences whose tail holds W uncompressed tokens in FULL blocks, the last (possibly partial) block
 *          excluded (App. C.4): t = seq_len mod block_size, eligible iff uncompressed - t >= W; window start
 *          h = seq_len - t - W.  The first max_select eligible sequences in batch order are taken (the paper takes "30
 *          sequences", L275, and does not say which: reading G18).
 *          For selected sequence number x: sel_ids[x] = s, sel_win_start[x] = h, sel_seq_lens[x] = seq_len,
 *          sel_block_table[x][:] = block_table[s][:].  Rows x >= *sel_count get sel_ids = -1, sel_seq_lens = -1.
 * `uncompressed` is the number of trailing tokens never compressed (buffer and partial block included); the paper's
 * per-sequence variable "reset to 0 after each compression" (L354) counts the tokens beyond the compressed window, i.e.
 * this counter minus the U + t tokens that kara_oracle_policy_commit leaves in it.  active may be NULL (all active). */
int kara_oracle_policy_step(int n_seqs, int max_blocks, int block_size, int32_t* block_table, int32_t* seq_lens,
                            int32_t* uncompressed, const uint8_t* active, int32_t* free_list, int32_t* free_count,
                            int32_t* step_counter, int delta, int W, int max_select,
                            int32_t* sel_ids, int32_t* sel_count, int32_t* sel_block_table, int32_t* sel_seq_lens,
                            int32_t* sel_win_start, int32_t* exhausted);

/* After the selected sub-batch has been compressed and committed (kara_oracle_compress_window on sel_block_table /
 * sel_seq_lens / sel_win_start): UpdateMetadata of the running queue (Alg. 1 l.12): for x < sel_count, s = sel_ids[x]:
 * block_table[s][:] = sel_block_table[x][:], seq_lens[s] = sel_seq_lens[x] (= h + keep + U + t), and the counter of
 * uncompressed trailing tokens becomes U + t, t = new seq_len - (sel_win_start[x] + keep + U). */
int kara_oracle_policy_commit(int max_blocks, const int32_t* sel_ids, int sel_count, const int32_t* sel_block_table,
                              const int32_t* sel_seq_lens, const int32_t* sel_win_start, int keep, int U,
                              int32_t* block_table, int32_t* seq_lens, int32_t* uncompressed);

/* Window-query producer (App. C.2: at each compression "we run an additional forward pass on the tokens
 * in the current window ... we compute only the query projections, ..."): the query states of T window tokens
 * of one layer from their (normalised) hidden states,
 *     q[t][h][:] = RoPE_{pos[t]}( sum_k hidden[t][k] * wq[h d + :][k] )
 * bf16 inputs widened, products and sums in double, rounded ONCE to bf16 (round to nearest even).  Reading G19:
 * rotary embedding in the rotate-half pairing of the paper's models (Llama / Qwen): for c < d/2, f_c = theta^(-2c/d),
 * a = pos f_c:  out[c] = q[c] cos a - q[c+d/2] sin a,  out[c+d/2] = q[c+d/2] cos a + q[c] sin a;  no bias, no q-norm.
 * positions == NULL: no rotary embedding.  hidden [T][d_model], wq [n_q_heads*d][d_model], out [T][n_q_heads][d] (bf16 bits). */
int kara_oracle_window_queries(const uint16_t* hidden, const uint16_t* wq, const int32_t* positions, double rope_theta,
                               int T, int d_model, int n_q_heads, int d, uint16_t* out);

#ifdef __cplusplus
}
#endif
#endif /* KARA_ORACLE_H */
