// policy.cu — the periodic compression policy on the device (Alg. 1, reconstructed per DESIGN.md reading
// G12; App. C.4; B.1, L275): the bookkeeping of one decoding step for the running queue, so that the library is a
// drop-in cache manager:
//   policy_step_kernel   l.2  one generated token per active sequence: a token at a block boundary pops a block from the TOP
//                             of the free-list stack (batch order: exclusive scan, no atomics, so the result is bit-comparable
//                             with the oracle's sequential loop); seq_len += 1, uncompressed += 1
//                        l.3  g += 1
//                        l.4-5 if g > W and g mod delta == 0: SELECT the first max_select sequences (batch order) whose tail
//                             holds W uncompressed tokens in full blocks, the partial last block excluded (App. C.4); their
//                             block-table rows, lengths and window starts are gathered into a dense sub-batch that
//                             kara_compress_window takes as it is (rows past the count are marked absent: seq_len = -1)
//   policy_commit_kernel l.12 UpdateMetadata of the running queue from the compressed sub-batch; the counter of never-compressed
//                             trailing tokens becomes U + t (reading G18)
// One CTA: the work is a few integers per sequence.
#include "kara_internal.h"

namespace kara {

namespace {

constexpr int kThreads = 256;

// exclusive scan of one int per thread over the block; total in *total.  Ends synchronised.
__device__ __forceinline__ int block_scan(int v, int* warp_tot, int* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int y = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += y;
  }
  __syncthreads();
  if (lane == 31) warp_tot[warp] = inc;
  __syncthreads();
  int base = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < kThreads / 32; ++w) {
    const int x = warp_tot[w];
    if (w < warp) base += x;
    tot += x;
  }
  *total = tot;
  return base + inc - v;
}

struct PolicyArgs {
  int n_seqs, max_blocks, bs, bs_log2, delta, W, max_select;
  int32_t* block_table; int32_t* seq_lens; int32_t* uncompressed; const uint8_t* active;
  int32_t* free_list; int32_t* free_count; int32_t* step_counter;
  int32_t* sel_ids; int32_t* sel_count; int32_t* sel_block_table; int32_t* sel_seq_lens; int32_t* sel_win_start;
  int32_t* exhausted;
};

__global__ void __launch_bounds__(kThreads) policy_step_kernel(const PolicyArgs a) {
  __shared__ int warp_tot[kThreads / 32];
  __shared__ int s_run;
  const int tid = threadIdx.x;
  // ---- l.2: one generated token per active sequence; block allocation in batch order ----
  const int fc0 = *a.free_count;
  if (tid == 0) s_run = 0;
  __syncthreads();
  int n_exh = 0;
  for (int s0 = 0; s0 < a.n_seqs; s0 += kThreads) {
    const int s = s0 + tid;
    const bool act = s < a.n_seqs && (!a.active || a.active[s]);
    const int len = act ? a.seq_lens[s] : 0;
    const bool need = act && (len & (a.bs - 1)) == 0;                    // the token opens a new block
    const int b = len >> a.bs_log2;
    const bool can = need && b < a.max_blocks;                           // (a full table row never pops)
    int tot;
    const int rank = s_run + block_scan(can ? 1 : 0, warp_tot, &tot);    // pops before this sequence, batch order
    bool advance = act;
    if (need) {
      if (can && rank < fc0) a.block_table[(long long)s * a.max_blocks + b] = a.free_list[fc0 - 1 - rank];
      else { advance = false; ++n_exh; }
    }
    if (advance) { a.seq_lens[s] = len + 1; a.uncompressed[s] += 1; }
    __syncthreads();
    if (tid == 0) s_run += tot;
    __syncthreads();
  }
  if (n_exh) atomicAdd(a.exhausted, n_exh);                               // a count: order-free
  __syncthreads();
  const int pops = min(s_run, fc0);                                       // blocks taken off the stack in this step
  __syncthreads();
  // ---- l.3 ----
  const int g = *a.step_counter + 1;
  // ---- l.4-5: SELECT ----
  const bool event = g > a.W && g % a.delta == 0;
  if (tid == 0) s_run = 0;
  __syncthreads();
  if (event) {
    for (int s0 = 0; s0 < a.n_seqs; s0 += kThreads) {
      const int s = s0 + tid;
      const bool act = s < a.n_seqs && (!a.active || a.active[s]);
      const int len = act ? a.seq_lens[s] : 0;
      const int t = len & (a.bs - 1);                                    // the last (possibly partial) block is excluded
      const bool elig = act && a.uncompressed[s] - t >= a.W;
      int tot;
      const int x = s_run + block_scan(elig ? 1 : 0, warp_tot, &tot);
      if (elig && x < a.max_select) { a.sel_ids[x] = s; a.sel_win_start[x] = len - t - a.W; a.sel_seq_lens[x] = len; }
      __syncthreads();
      if (tid == 0) s_run += tot;
      __syncthreads();
    }
  }
  const int cnt = min(s_run, a.max_select);
  for (int x = cnt + tid; x < a.max_select; x += kThreads) { a.sel_ids[x] = -1; a.sel_seq_lens[x] = -1; a.sel_win_start[x] = 0; }
  __syncthreads();
  for (int x = 0; x < a.max_select; ++x) {
    const int s = x < cnt ? a.sel_ids[x] : -1;
    for (int b = tid; b < a.max_blocks; b += kThreads)
      a.sel_block_table[(long long)x * a.max_blocks + b] = s >= 0 ? a.block_table[(long long)s * a.max_blocks + b] : -1;
  }
  if (tid == 0) {
    *a.sel_count = cnt;
    *a.step_counter = g;
    *a.free_count = fc0 - pops;
  }
}

struct CommitArgs {
  int max_select, max_blocks, keep, U, W;
  const int32_t* sel_ids; const int32_t* sel_count; const int32_t* sel_block_table; const int32_t* sel_seq_lens;
  const int32_t* sel_win_start;
  int32_t* block_table; int32_t* seq_lens; int32_t* uncompressed;
};

__global__ void __launch_bounds__(kThreads) policy_commit_kernel(const CommitArgs a) {
  __shared__ int s_skip;
  const int cnt = min(*a.sel_count, a.max_select);
  for (int x = 0; x < cnt; ++x) {
    const int s = a.sel_ids[x];
    if (s < 0) continue;
    // A sub-batch row that kara_compress_window skipped (a fault recorded in its status word) comes back with the length
    // it went in with — a compressed one is shorter by W - keep - U > 0 tokens.  Such a sequence was not compressed:
    // its table row, length and uncompressed count stay as they are (it is still eligible at the next event).
    if (threadIdx.x == 0) s_skip = (a.sel_seq_lens[x] == a.seq_lens[s] && a.keep + a.U < a.W) ? 1 : 0;
    __syncthreads();
    if (!s_skip) {
      for (int b = threadIdx.x; b < a.max_blocks; b += kThreads)
        a.block_table[(long long)s * a.max_blocks + b] = a.sel_block_table[(long long)x * a.max_blocks + b];
      if (threadIdx.x == 0) {
        const int len = a.sel_seq_lens[x];
        a.seq_lens[s] = len;
        a.uncompressed[s] = a.U + (len - (a.sel_win_start[x] + a.keep + a.U));   // buffer + tail stay uncompressed
      }
    }
    __syncthreads();
  }
}

}  // namespace

cudaError_t launch_policy_step(int n_seqs, int max_blocks, int bs, int bs_log2, int delta, int W, int max_select,
                               int32_t* block_table, int32_t* seq_lens, int32_t* uncompressed, const uint8_t* active,
                               int32_t* free_list, int32_t* free_count, int32_t* step_counter, int32_t* sel_ids,
                               int32_t* sel_count, int32_t* sel_block_table, int32_t* sel_seq_lens, int32_t* sel_win_start,
                               int32_t* exhausted, cudaStream_t st) {
  PolicyArgs a{n_seqs, max_blocks, bs, bs_log2, delta, W, max_select, block_table, seq_lens, uncompressed, active,
               free_list, free_count, step_counter, sel_ids, sel_count, sel_block_table, sel_seq_lens, sel_win_start,
               exhausted};
  policy_step_kernel<<<1, kThreads, 0, st>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_policy_commit(int max_select, int max_blocks, int keep, int U, int W, const int32_t* sel_ids,
                                 const int32_t* sel_count, const int32_t* sel_block_table, const int32_t* sel_seq_lens,
                                 const int32_t* sel_win_start, int32_t* block_table, int32_t* seq_lens,
                                 int32_t* uncompressed, cudaStream_t st) {
  CommitArgs a{max_select, max_blocks, keep, U, W, sel_ids, sel_count, sel_block_table, sel_seq_lens, sel_win_start,
               block_table, seq_lens, uncompressed};
  policy_commit_kernel<<<1, kThreads, 0, st>>>(a);
  return cudaGetLastError();
}

}  // namespace kara
