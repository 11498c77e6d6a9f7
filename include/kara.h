/*
 * kara.h — C ABI of libkara: Kara's decoding-time sliding-window KV-cache compression step
 * (arxiv/paper_2607_01237) on a paged bf16 KV cache, as hand-written CUDA for sm_100a (B200).
 *
 * What one kara_compress_window call computes, for every (sequence, layer, KV head) "unit"
 * of the batch (window-relative 0-based positions; W = |W| window length, U = |U| protected
 * buffer at the window's end, n = W-U compressible keys, G = n_q_heads / n_kv_heads):
 *
 *   a1 score      A_j = sum_{i<W} sum_{g<G} softmax_j( Q[(i,g)] . K[j] / sqrt(d) )      j in [0,n)
 *                 PAPER.md Eq. 4 (L115): bidirectional (unmasked) attention of ALL window
 *                 queries against the compressible keys, softmax over keys, colsum over queries.
 *   a2 top-k      I = the k = keep - alpha best-scoring positions, keep = ceil(r n)
 *                 PAPER.md Eq. 5 (L117).
 *   a3 Token2Chunk consecutive members a<b of sorted I are chunk endpoints; eligible iff
 *                 b-a < gamma; R = (A_a + A_b)(b-a-1); the floor(alpha/(gamma-2)) best eligible
 *                 chunks add their interiors; the rest of the budget is filled with the best
 *                 unselected positions                    PAPER.md Eq. 6-8 (L133-138), App. C.3 (L350).
 *   a4 compaction (K,V)[h .. h+keep) <- (K,V)[h + F[.]], buffer + tail rows follow directly;
 *                 rows [0,h) are never touched          PAPER.md Eq. 9 (L142), Sec. 4.3 (L150).
 *   a5 metadata   seq_len <- h+keep+U+t; trailing blocks of the block table are pushed on the
 *                 device free list and set to -1         PAPER.md Alg. 1 l.11-12 (L336-337), App. C.4 (L354).
 *
 * Tie-breaks and the other places where the paper is silent follow DESIGN.md "Readings":
 * GQA heads are summed (G1); ties -> lower index first (G4); keep = ceil(ratio*n - 1e-9) with
 * ratio a double (G5); chunk filter before top-P (G7); retained rows keep ascending order (G10).
 *
 * Conventions.  Pointers marked [dev] are device memory OWNED BY THE CALLER (e.g. torch
 * tensors); [host] are host memory.  The library allocates nothing on the device except through
 * kara_compress_window_host's internal staging buffers; its device image carries two static arrays on every GPU
 * that loads it (1 MiB of rotary tables for kara_window_queries_static, 128 KiB of per-handle status words).
 * Calls are asynchronous on `stream`
 * (a cudaStream_t passed as void*; NULL = legacy default stream) unless marked synchronous.
 * Every call returns 0 (KARA_OK) or a negative KARA_E* code and never throws or aborts;
 * kara_last_error() gives a thread-local message for the last failure.  Data-dependent faults
 * found on the device (a block id outside the pool, a sequence shorter than its window) set bits
 * in a device status word and the offending SEQUENCE is skipped as a whole: every block-table entry
 * its window touches is validated before anything is written, so its K/V rows, its block-table row,
 * its seq_len and the free list stay byte-identical (its debug scores / indices are undefined).  The
 * check depends on the tables only, so every layer-range call and the committing call skip the same
 * sequences.  The status word accumulates over the calls of one handle until kara_status() reads it.
 *
 * Physical layout fixed by kara_init_cache (separate K and V pools, each):
 *     bf16 pool[n_layers][num_blocks][n_kv_heads][block_size][head_dim]
 * so one (layer, block, kv_head) tile is block_size*head_dim*2 contiguous bytes (one TMA box
 * per 64-element column panel).  Logical token p of sequence s lives in block
 * block_table[s][p / block_size], slot p % block_size, for every layer and head.
 */
#ifndef KARA_H
#define KARA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define KARA_OK 0
#define KARA_EINVAL (-1)       /* bad argument / shape / null pointer */
#define KARA_EBUDGET (-2)      /* keep - alpha < 1, keep > n, or gamma < 3 */
#define KARA_EUNSUPPORTED (-3) /* head_dim not in {64,128}, block_size not a power of two in [16,256], n > 2048 */
#define KARA_ECUDA (-4)        /* a CUDA call or launch failed (message in kara_last_error) */
#define KARA_ENOMEM (-5)       /* workspace too small */

/* flags of kara_compress_window */
#define KARA_COMMIT 1u           /* run a5 (seq_lens, block table truncation, free list) after a4.
                                    Set it only on the call that finishes the LAST layer: blocks must
                                    not be freed while other layers still hold live rows in them. */
#define KARA_KEEP_DEBUG 2u       /* keep scores / I / F of every unit in the workspace for kara_gather_debug */
#define KARA_SCORE_QBUF_ONLY 4u  /* ablation "w/o Bi-Attention": queries = buffer U only */
#define KARA_SCORE_SIMT 8u       /* run the CUDA-core score kernel (debug cross-check of the tcgen05 path).  It is never
                                    chosen for you: a call the tcgen05 kernel cannot take (no sm_100 device, a K pool of
                                    2^31 rows or more, 2^31 window tokens or more) returns KARA_EUNSUPPORTED without it */

/* `what` of kara_gather_debug */
#define KARA_DBG_K_LOGICAL 0  /* bf16 [seq_len][d] rows of (layer, seq, kv_head) read through the block table */
#define KARA_DBG_V_LOGICAL 1
#define KARA_DBG_SCORES 2     /* fp32 [n]      last call with KARA_KEEP_DEBUG */
#define KARA_DBG_IDX_TOPK 3   /* int32 [k]     ascending (Eq. 5) */
#define KARA_DBG_IDX_FINAL 4  /* int32 [keep]  ascending (Eq. 8 + C.3) */
#define KARA_DBG_BLOCK_TABLE_ROW 5 /* int32 [max_blocks] */
#define KARA_DBG_FREE_LIST 6  /* int32 [free_count] */

/* bits of the device status word */
#define KARA_ST_BAD_BLOCK 1   /* a block-table entry touched by the window is outside [0, num_blocks) */
#define KARA_ST_SHORT_SEQ 2   /* win_start < 0 or win_start + W > seq_len */
#define KARA_ST_TABLE_OVERFLOW 4 /* ceil(seq_len / block_size) > max_blocks */
#define KARA_ST_FREE_OVERFLOW 8  /* a5 would push past free_list[num_blocks) (stale, negative or duplicated free_count): the
                                    K/V rows are already compacted at that point, so seq_lens and the block tables ARE
                                    committed (they must describe the rows as they now lie), but the blocks the step frees
                                    are dropped instead of pushed and free_count does not move — per group of 256 sequences
                                    in batch order.  The cache stays consistent; the blocks leak until the caller rebuilds
                                    its free list.  (The other three bits skip the sequence as a whole.) */

typedef struct kara_cache kara_cache;

/* Fix the geometry of the paged cache.  Returns a handle (host object, no device allocation) or
 * NULL (kara_last_error says why: KARA_EUNSUPPORTED shapes).  PAPER.md:L82 (PagedAttention blocks). */
kara_cache* kara_init_cache(int block_size, int n_layers, int n_kv_heads, int head_dim);

/* Frees the handle and any staging buffers kara_compress_window_host allocated.  Synchronous. */
void kara_destroy(kara_cache* c);

/* Bytes of one pool (K or V) with num_blocks blocks, and of one block across all layers' slices. */
int64_t kara_pool_bytes(const kara_cache* c, int64_t num_blocks);
int64_t kara_block_bytes(const kara_cache* c);

/* Attach caller-owned device memory: the two pools (layout above, 256-byte aligned) and the
 * free list: free_list [dev int32 num_blocks] is a stack whose first *free_count entries are the
 * free block ids; a5 appends to it.  Must be called before kara_compress_window.  Synchronous
 * (builds the TMA descriptor of the K pool). */
int kara_attach_pool(kara_cache* c, void* k_pool /*dev*/, void* v_pool /*dev*/, int64_t num_blocks,
                     int32_t* free_list /*dev*/, int32_t* free_count /*dev [1]*/);

/* keep = ceil(ratio * n) evaluated as (int)ceil(ratio*n - 1e-9) (reading G5); <0 on bad input. */
int kara_budget(int n, double ratio);

/* Bytes of device scratch kara_compress_window needs for this geometry. */
size_t kara_workspace_bytes(const kara_cache* c, int n_layers_in_call, int n_seqs, int n_q_heads,
                            int W, int U, double ratio, int alpha);

/* The batched compression step: a1-a4 for layers [layer_begin, layer_end) x n_seqs sequences x
 * all KV heads, and a5 if flags & KARA_COMMIT.
 *   block_table [dev int32 n_seqs x max_blocks] in/out   -1 padded; freed entries become -1
 *   seq_lens    [dev int32 n_seqs]              in/out   tokens currently stored per sequence
 *   win_start   [dev int32 n_seqs] or NULL      in       h: first token of the window; NULL => seq_len - W.
 *                                                        t = seq_len - h - W tail tokens (App. C.4's partial
 *                                                        last block) are carried over behind the buffer.
 *   window_q    [dev bf16 (layer_end-layer_begin) x n_seqs x W x n_q_heads x head_dim]  in
 *                                                        query states of the window tokens,
 *                                                        16-byte aligned
 *   ratio, alpha, gamma                                  r, chunk budget, max chunk length (Eq. 5-7)
 *   workspace   [dev] >= kara_workspace_bytes(...), 256-byte aligned; contents are scratch
 * All sequences share W, U, ratio, alpha, gamma.  After the call the last U tokens of
 * the old window are the first U uncompressed tokens behind the retained ones. */
int kara_compress_window(kara_cache* c, int layer_begin, int layer_end, int n_seqs,
                         int32_t* block_table /*dev*/, int max_blocks, int32_t* seq_lens /*dev*/,
                         const int32_t* win_start /*dev or NULL*/, const void* window_q /*dev*/,
                         int n_q_heads, int W, int U, double ratio, int alpha, int gamma,
                         unsigned flags, void* workspace /*dev*/, size_t workspace_bytes,
                         void* stream);

/* Prefill / multi-window batch (App. C.2: "partition the prompt into multiple windows of length |W| and
 * perform window-wise compression ... in parallel"; L346).  Reading G17: the n_windows windows of a sequence
 * are the disjoint ranges [h + w W, h + (w+1) W), h = win_start[s] (NULL => seq_len - n_windows*W); each is scored with its
 * own W queries against its own n keys and selected on its own (a1-a3 unchanged); a4 lays the retained rows and the buffer
 * of window w down behind those of window w-1 and the t = seq_len - h - n_windows*W tail rows behind the last window:
 *     new[h + w (keep+U) + c]        = old[h + w W + F_w[c]]    c < keep
 *     new[h + w (keep+U) + keep + c] = old[h + w W + n + c]     c < U
 *     new[h + n_windows (keep+U) + c] = old[h + n_windows W + c]   c < t
 * a5: seq_len <- h + n_windows (keep+U) + t.  window_q is [layers x n_seqs x n_windows*W x n_q_heads x head_dim]; the
 * workspace must hold kara_workspace_bytes(..., n_seqs * n_windows, ...) bytes; after such a call the `seq` argument of
 * kara_gather_debug(SCORES / IDX_*) is sequence * n_windows + window.  n_windows = 1 is kara_compress_window. */
int kara_compress_windows(kara_cache* c, int layer_begin, int layer_end, int n_seqs,
                          int32_t* block_table /*dev*/, int max_blocks, int32_t* seq_lens /*dev*/,
                          const int32_t* win_start /*dev or NULL*/, int n_windows, const void* window_q /*dev*/,
                          int n_q_heads, int W, int U, double ratio, int alpha, int gamma,
                          unsigned flags, void* workspace /*dev*/, size_t workspace_bytes, void* stream);

/* Same step with HOST buffers for everything but the resident pools: copies window_q,
 * block_table, seq_lens, win_start host->device into library-owned staging buffers, runs
 * kara_compress_window on `stream`, copies block_table and seq_lens back and reports the new
 * free count.  Synchronous on return.  Host buffers should be pinned for full copy bandwidth. */
int kara_compress_window_host(kara_cache* c, int layer_begin, int layer_end, int n_seqs,
                              int32_t* block_table /*host in/out*/, int max_blocks,
                              int32_t* seq_lens /*host in/out*/, const int32_t* win_start /*host or NULL*/,
                              const void* window_q /*host*/, int n_q_heads, int W, int U, double ratio,
                              int alpha, int gamma, unsigned flags, int32_t* free_count_out /*host [1] or NULL*/,
                              void* stream);

/* Synchronous read-back for tests: writes up to out_capacity_bytes to `out` [host] and the
 * number of ELEMENTS written to *out_count.  SCORES / IDX_* refer to the unit (layer, seq, kv_head)
 * of the last kara_compress_window call made with KARA_KEEP_DEBUG (layer is absolute). */
int kara_gather_debug(kara_cache* c, int what, int layer, int seq, int kv_head,
                      const int32_t* block_table /*dev*/, const int32_t* seq_lens /*dev*/,
                      int max_blocks, void* out /*host*/, int64_t out_capacity_bytes,
                      int64_t* out_count /*host*/);

/* Periodic compression policy on the device (Alg. 1, as reconstructed by DESIGN.md reading G12;
 * App. C.4; B.1, L275): the bookkeeping of ONE decoding step of the running queue, asynchronous on `stream`.
 *   l.2   every active sequence has generated one token (the caller's decode step writes its K/V row): a token at a block
 *         boundary takes a block from the TOP of the attached free-list stack, sequences in batch order (reading G18);
 *         seq_len += 1, uncompressed += 1.  A sequence that needs a block while the stack is empty (or its table row is
 *         full) is not advanced and *exhausted is incremented — preemption is the serving engine's business.
 *   l.3   *step_counter += 1  (= g)
 *   l.4-5 if g > W and g mod delta == 0: SELECT the first max_select sequences, in batch order, whose tail holds W
 *         uncompressed tokens in full blocks — t = seq_len mod block_size tokens of the partial last block are excluded
 *         (App. C.4): eligible iff uncompressed - t >= W; window start h = seq_len - t - W.  Selected sequence number x
 *         gets sel_ids[x] = s, sel_win_start[x] = h, sel_seq_lens[x] = seq_len, sel_block_table[x][:] = block_table[s][:];
 *         rows x >= *sel_count get sel_ids = -1, sel_seq_lens = -1 ("absent": kara_compress_window skips them silently).
 * The sel_* arrays ARE the sub-batch of the compression event: recompute the window queries of the selected sequences
 * (sub-batch order), call kara_compress_window(n_seqs = max_select, sel_block_table, sel_seq_lens, sel_win_start, ...,
 * KARA_COMMIT), then kara_policy_commit.  `uncompressed` [dev int32 n_seqs] counts the trailing tokens never compressed
 * (buffer and partial block included: the paper's per-sequence variable, L354, counts the tokens beyond the last window,
 * i.e. this minus U + t).  active [dev uint8 n_seqs] or NULL (all).  All sel_* are [dev], sized max_select
 * (sel_block_table: max_select x max_blocks); step_counter, sel_count, exhausted are [dev int32 1]. */
int kara_policy_step(kara_cache* c, int n_seqs, int32_t* block_table /*dev, in/out*/, int max_blocks,
                     int32_t* seq_lens /*dev, in/out*/, int32_t* uncompressed /*dev, in/out*/,
                     const uint8_t* active /*dev or NULL*/, int32_t* step_counter /*dev*/, int delta, int W,
                     int max_select, int32_t* sel_ids, int32_t* sel_count, int32_t* sel_block_table,
                     int32_t* sel_seq_lens, int32_t* sel_win_start, int32_t* exhausted, void* stream);

/* Alg. 1 l.12 UpdateMetadata(e) for the running queue after the sub-batch was compressed and committed: for x < *sel_count,
 * s = sel_ids[x]: block_table[s][:] = sel_block_table[x][:], seq_lens[s] = sel_seq_lens[x], and uncompressed[s] = U + t with
 * t = sel_seq_lens[x] - (sel_win_start[x] + keep + U), keep = ceil(ratio (W-U)).  A row whose sel_seq_lens[x] still equals
 * seq_lens[s] although keep + U < W was skipped by kara_compress_window (a fault in its status word): nothing of that
 * sequence is committed, it stays eligible.  Asynchronous on `stream`. */
int kara_policy_commit(kara_cache* c, int max_select, const int32_t* sel_ids, const int32_t* sel_count,
                       const int32_t* sel_block_table, const int32_t* sel_seq_lens, const int32_t* sel_win_start,
                       int W, int U, double ratio, int32_t* block_table /*dev*/, int max_blocks,
                       int32_t* seq_lens /*dev*/, int32_t* uncompressed /*dev*/, void* stream);

/* Window-query producer (App. C.2: at each compression the window's query states are recomputed — "we compute
 * only the query projections, the causal attention against the cached prefix KV states, and the FFN").  This is
 * the projection step for ONE layer, written directly in the layout kara_compress_window reads:
 *     window_q_out[t][h][:] = RoPE_{positions[t]}( hidden[t][:] . wq[h*head_dim + :][:]^T )      bf16 in / out, fp32 accumulate
 * Reading G19: rotary embedding in the rotate-half pairing of the paper's models — for c < d/2, f_c = theta^(-2c/d),
 * a = pos f_c: out[c] = q[c] cos a - q[c+d/2] sin a, out[c+d/2] = q[c+d/2] cos a + q[c] sin a — no bias, no q-norm; the hidden
 * states (the layer's normalised inputs, i.e. everything before the projection) are the caller's.
 *   hidden        [dev bf16 n_tokens x d_model]   d_model a multiple of 64; 16-byte aligned
 *   wq            [dev bf16 (n_q_heads*head_dim) x d_model]
 *   positions     [dev int32 n_tokens] in [0, max_position], or NULL: no rotary embedding.  The range is the CALLER'S
 *                 contract: there is no device-side check and no status word on this call — a position outside it is
 *                 rotated by the angle of some position inside it (the table index is clamped), i.e. wrongly and silently
 *   window_q_out  [dev bf16 n_tokens x n_q_heads x head_dim]  (tokens in the order of the call's window_q: sequence, token)
 *   workspace     [dev] >= kara_window_queries_workspace_bytes(max_position, head_dim) (cos / sin tables; unused without positions).
 *                 The tables are rebuilt on `stream` by every call (a few microseconds), so calls that may overlap on the GPU
 *                 must not share a workspace
 * Asynchronous on `stream`.  One hand-written tcgen05 / TMA GEMM with the rotary embedding fused into its epilogue. */
size_t kara_window_queries_workspace_bytes(int max_position, int head_dim);
int kara_window_queries(const void* hidden /*dev*/, const void* wq /*dev*/, const int32_t* positions /*dev or NULL*/,
                        int max_position, double rope_theta, int n_tokens, int d_model, int n_q_heads, int head_dim,
                        void* window_q_out /*dev*/, void* workspace /*dev*/, size_t workspace_bytes, void* stream);

/* kara_window_queries for callers that cannot bring a workspace: the rotary cos / sin tables go into an array that is part
 * of libkara's own device image instead of into caller memory.  Everything else — arguments, layouts, arithmetic, kernels,
 * result bits — is kara_window_queries.
 *
 * Who needs it.  The producer runs inside a compression event in the middle of decoding.  A serving engine has by then
 * given every byte of HBM that was left after the weights to its paged KV pool, so a cudaMalloc at that point fails; where
 * it would still succeed it stalls the whole device while the driver maps memory, which no other stream's decode step can
 * afford; and engines that route all device memory through one pool (so that usage stays accountable) do not let a
 * library call the CUDA allocator behind their back.  Such a caller may also have no spare pool buffer to lend for the
 * few hundred KB of tables.  This entry point calls no cudaMalloc, cudaFree or other allocating routine, ever.
 *
 * The limit.  The array is KARA_STATIC_SCRATCH_BYTES (1 MiB) and every GPU on which the process uses libkara carries it from
 * the moment the library's device code is loaded there until the process exits.  The tables take
 * kara_window_queries_workspace_bytes(max_position, head_dim) bytes, so max_position <= 458,751 fits at head_dim 128 and
 * <= 983,039 at head_dim 64.  A larger max_position is refused with KARA_ENOMEM before anything is launched (the message
 * names the bytes needed and the limit); use kara_window_queries with your own workspace then.
 *
 * First call on a device.  The array's device address is looked up (cudaGetSymbolAddress) the first time the entry point
 * is called with a given device current, and remembered per device; a failure of that lookup is returned as KARA_ECUDA.
 * Make that first call during start-up, outside any stream capture.  Later calls on that device do no set-up.
 *
 * Sharing.  There is one array per GPU and every call on that GPU uses it.  Nothing in it has to start at zero and nothing
 * is carried from call to call: each call rewrites, on `stream`, every table row its own GEMM epilogue reads (for its own
 * theta, head_dim and max_position) before that kernel runs, and the previous call's tables are simply overwritten.  The
 * price is that two calls whose kernels can overlap on the GPU — different streams, or different host threads without an
 * event between them — race on the tables and may rotate with each other's angles.  Issue the calls of one GPU on one
 * stream or order them with events.  positions == NULL (no rotary embedding) touches no scratch at all.
 * Asynchronous on `stream`. */
#define KARA_STATIC_SCRATCH_BYTES 1048576
int kara_window_queries_static(const void* hidden /*dev*/, const void* wq /*dev*/, const int32_t* positions /*dev or NULL*/,
                               int max_position, double rope_theta, int n_tokens, int d_model, int n_q_heads,
                               int head_dim, void* window_q_out /*dev*/, void* stream);

/* Synchronous: reads and clears the device status word (0 = no fault).  The word is sticky: it holds the
 * OR of the faults of every kara_compress_window(s) call on this handle since the last kara_status() (or since
 * kara_attach_pool, which clears it) — whatever workspaces those calls used.  It lives in device memory that belongs to
 * the library (a slot of a static array, one per live handle, at most 4096 handles), not in the workspace. */
int kara_status(kara_cache* c, int32_t* status_out /*host*/);

/* Number of kernel launches the last kara_compress_window call made (for bench.py's gpu_launches). */
int kara_last_launch_count(const kara_cache* c);

/* Which score kernel the last call used: 0 = none yet, 1 = CUDA-core (SIMT), 2 = tcgen05/TMA. */
int kara_last_score_path(const kara_cache* c);
/* "" if the tcgen05 kernel ran, else why the CUDA-core kernel did (only ever: KARA_SCORE_SIMT was set).  The CUDA-core
 * kernel is a cross-check, not a second backend: bench.py refuses its numbers. */
const char* kara_last_score_path_reason(const kara_cache* c);

/* Device time of the score kernel (a1) alone: when enabled, every kara_compress_window call
 * brackets its score launch with CUDA events on `stream`; kara_score_kernel_ms() synchronises on
 * the last pair and returns its milliseconds (<0 if none).  Used for bench.py's roofline object. */
int kara_enable_score_timing(kara_cache* c, int enable);
float kara_score_kernel_ms(kara_cache* c);

/* Thread-local message for the last failing call on this thread ("" if none). */
const char* kara_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* KARA_H */
