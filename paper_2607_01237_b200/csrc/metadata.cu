// metadata.cu — a5: "UpdateMetadata" + block release (Alg. 1 l.12, L337; Sec. 4.3;
// App. C.4), and the logical-row gather behind kara_gather_debug.
//
// One CTA walks the sequences in batch order, 256 at a time: per sequence
//   new_len = h + NW (keep + U) + t,  new_nb = ceil(new_len / bs),  old_nb = ceil(len / bs)     (NW = windows per sequence)
// the freed counts are exclusive-scanned so that block_table[s][new_nb:old_nb] lands on the free
// list in sequence order, table order (reading G16: a deterministic scan, not atomics, so the
// list is bit-comparable with the oracle's).
#include "kara_internal.h"

namespace kara {

namespace {

constexpr int kThreads = 256;

__global__ void __launch_bounds__(kThreads) metadata_kernel(const Call c) {
  __shared__ int warp_tot[kThreads / 32];
  __shared__ int s_running;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  asm volatile("griddepcontrol.wait;" ::: "memory");   // launched programmatically behind select_compact
  if (tid == 0) s_running = *c.free_count;
  __syncthreads();
  for (int s0 = 0; s0 < c.n_seqs; s0 += kThreads) {
    const int s = s0 + tid;
    int freed = 0, new_nb = 0, old_nb = 0, new_len = 0;
    bool ok = false;
    if (s < c.n_seqs) {
      const int len = c.seq_lens[s];
      const int h = c.win_start ? c.win_start[s] : len - c.n_windows * c.W;
      const int t = len - h - c.n_windows * c.W;
      old_nb = (len + c.g.bs - 1) >> c.g.bs_log2;
      ok = (len >= 0 && h >= 0 && t >= 0 && old_nb <= c.max_blocks);   // len < 0: absent row of a policy sub-batch
      if (ok) {
        // the same validation select_compact ran: a sequence with a block id outside the pool in its window
        // was not compacted and is not committed (its table row, seq_len and the free list stay as they are)
        const int32_t* row = c.block_table + (long long)s * c.max_blocks;
        for (int b = h >> c.g.bs_log2; b < old_nb; ++b) ok &= (row[b] >= 0 && row[b] < c.g.num_blocks);
        if (!ok) atomicOr(c.status, KARA_ST_BAD_BLOCK);
      }
      if (ok) {
        new_len = h + c.n_windows * (c.keep + c.U) + t;   // every window leaves keep + U rows behind
        new_nb = (new_len + c.g.bs - 1) >> c.g.bs_log2;
        freed = old_nb - new_nb;
      }
    }
    int inc = freed;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int y = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += y;
    }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    int base = s_running, tot = 0;
#pragma unroll
    for (int w = 0; w < kThreads / 32; ++w) {
      if (w < warp) base += warp_tot[w];
      tot += warp_tot[w];
    }
    base += inc - freed;
    // A stale or duplicated free_count must not push past the list.  By now a4 has already compacted the rows of these
    // sequences, so refusing the commit would leave seq_lens and the tables describing rows that no longer exist:
    // the lengths and tables ARE committed, but the trailing blocks of this group of 256 sequences are dropped instead
    // of pushed (they leak until the caller rebuilds its free list), free_count does not move, and the status word
    // says why.  The decision is uniform over the group, so the running count stays consistent.
    const bool overflow = (long long)s_running + tot > c.g.num_blocks || s_running < 0;
    if (overflow) {
      if (tid == 0) atomicOr(c.status, KARA_ST_FREE_OVERFLOW);
      tot = 0;
    }
    if (ok) {
      int32_t* row = c.block_table + (long long)s * c.max_blocks;
      for (int b = new_nb; b < old_nb; ++b) {
        if (!overflow) c.free_list[base + (b - new_nb)] = row[b];
        row[b] = -1;
      }
      c.seq_lens[s] = new_len;
    }
    __syncthreads();
    if (tid == 0) s_running += tot;
    __syncthreads();
  }
  if (tid == 0) *c.free_count = s_running;
}

__global__ void gather_rows_kernel(Geom g, const __nv_bfloat16* pool, int layer, int kv_head,
                                   const int32_t* bt_row, int length, __nv_bfloat16* out, int32_t* status) {
  const int vpr = g.d / 8;
  const long long total = (long long)length * vpr;
  for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < total;
       x += (long long)gridDim.x * blockDim.x) {
    const int pos = (int)(x / vpr), v = (int)(x % vpr);
    const int blk = bt_row[pos >> g.bs_log2];
    uint4 val = make_uint4(0, 0, 0, 0);
    if (blk < 0 || blk >= g.num_blocks) {
      atomicOr(status, KARA_ST_BAD_BLOCK);
    } else {
      const long long off = (long long)layer * g.sL + (long long)blk * g.sB + (long long)kv_head * g.sH +
                            (long long)(pos & (g.bs - 1)) * g.d;
      val = *reinterpret_cast<const uint4*>(pool + off + v * 8);
    }
    reinterpret_cast<uint4*>(out)[x] = val;
  }
}

}  // namespace

cudaError_t launch_metadata(const Call& c, cudaStream_t st) {
  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  cfg.gridDim = dim3(1); cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = 0; cfg.stream = st;
  return cudaLaunchKernelEx(&cfg, metadata_kernel, c);
}

cudaError_t launch_gather_rows(const Geom& g, const __nv_bfloat16* pool, int layer, int kv_head,
                               const int32_t* bt_row, int length, __nv_bfloat16* out, int32_t* status,
                               cudaStream_t st) {
  if (length <= 0) return cudaSuccess;
  const long long total = (long long)length * (g.d / 8);
  const int blocks = (int)((total + 255) / 256 > 1024 ? 1024 : (total + 255) / 256);
  gather_rows_kernel<<<blocks, 256, 0, st>>>(g, pool, layer, kv_head, bt_row, length, out, status);
  return cudaGetLastError();
}

}  // namespace kara
