// select_compact.cu — a2 + a3 + a4 for one (sequence, layer, KV head) unit per CTA.
//
//   a2  Eq. 5   I = top-(keep-alpha) of A under (A desc, index asc)
//   a3  Eq. 6-8 (L133-138) + App. C.3 (L350): eligible chunks (b-a < gamma, interior >= 1),
//       R = fl32(fl32(A_a + A_b) * gap), top-P under (R desc, ordinal asc), interiors added,
//       budget filled with the best unselected positions under (A desc, index asc)
//   a4  Eq. 9 (L142): rows h+F[c] -> h+c for K and V, buffer + tail rows behind them, in place
//
// Every TopK is the same block-wide primitive: an 8-bit-digit radix select over the
// order-preserving integer image of the fp32 key (4 passes, 256-bin shared-memory histogram,
// bins scanned by one warp with shuffles), then the tie class (key == threshold) is resolved in
// index order with a ballot-free segmented count + block scan.  All decisions are integer
// compares on fp32 bit patterns, so the result is a pure function of the scores.
//
// Prefill (n_windows > 1, App. C.2): the select kernel runs per (layer, sequence, window, head) unit and only
// writes F; compact_windows_kernel then moves the rows of ALL windows of a (layer, sequence, head) with one CTA, window by
// window, each window's retained rows + buffer laid down behind those of the window before it.
//
// In-place compaction is hazard-free with one CTA per unit: destination c <= source F[c] and both
// are increasing, so loading rows [c0,c1) into registers, barrier, then writing them never
// overwrites a row a later chunk still has to read.
#include "kara_internal.h"

namespace kara {

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
#ifndef KARA_SEL_VEC
#define KARA_SEL_VEC 4      // 16-byte vectors per thread and tensor in one compaction pass (measured: 4 x 5 CTAs/SM beats 8 x 3 at cfg4)
#endif
#ifndef KARA_SEL_OCC
#define KARA_SEL_OCC 5
#endif

struct Scratch {
  int hist[256];
  int warp_tot[kWarps];
  unsigned prefix, mask;
  int remaining;
  int bcast;
};

__device__ __forceinline__ unsigned key_of(float x) {
  const unsigned b = __float_as_uint(x);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

// exclusive scan of one int per thread over the block; returns the exclusive prefix, total in *total
__device__ __forceinline__ int block_excl_scan(int v, Scratch* sc, int* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int y = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += y;
  }
  __syncthreads();  // protect warp_tot from a previous use
  if (lane == 31) sc->warp_tot[warp] = inc;
  __syncthreads();
  int base = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < kWarps; ++w) {
    const int x = sc->warp_tot[w];
    if (w < warp) base += x;
    tot += x;
  }
  *total = tot;
  return base + inc - v;
}

// Marks sel[i] = 1 for the m best of the N candidates with valid(i), under (key desc, i asc).
// Requires 0 <= m <= #valid.  key/sel live in shared memory.  Block-wide; ends synchronised.
template <typename Valid>
__device__ void block_top_m(const unsigned* key, int N, int m, Valid valid, unsigned char* sel, Scratch* sc) {
  if (m <= 0) { __syncthreads(); return; }
  const int tid = threadIdx.x;
  if (tid == 0) { sc->prefix = 0u; sc->mask = 0u; sc->remaining = m; }
  for (int pass = 3; pass >= 0; --pass) {
    const int shift = pass * 8;
    sc->hist[tid] = 0;   // kThreads == 256 bins
    __syncthreads();
    const unsigned prefix = sc->prefix, mask = sc->mask;
    for (int i = tid; i < N; i += kThreads)
      if (valid(i) && (key[i] & mask) == prefix) atomicAdd(&sc->hist[(key[i] >> shift) & 255u], 1);
    __syncthreads();
    if (tid < 32) {
      // lane l owns bins 255-8l .. 248-8l (descending); find the bin where the running count
      // from the top first reaches `remaining`
      const int remaining = sc->remaining;
      int loc[8], sum = 0;
#pragma unroll
      for (int b = 0; b < 8; ++b) { loc[b] = sc->hist[255 - 8 * tid - b]; sum += loc[b]; }
      int inc = sum;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, inc, o);
        if (tid >= o) inc += y;
      }
      int above = inc - sum;  // candidates in strictly higher bins than this lane's
      if (above < remaining && inc >= remaining) {
#pragma unroll
        for (int b = 0; b < 8; ++b) {
          if (above + loc[b] >= remaining) {
            sc->prefix = prefix | ((unsigned)(255 - 8 * tid - b) << shift);
            sc->mask = mask | (255u << shift);
            sc->remaining = remaining - above;
            break;
          }
          above += loc[b];
        }
      }
    }
    __syncthreads();
  }
  // threshold key T = sc->prefix; everything above T is selected, plus the first `r` (index
  // order) of the tie class key == T
  const unsigned T = sc->prefix;
  const int r = sc->remaining;
  const int seg = (N + kThreads - 1) / kThreads;
  const int i0 = min(N, tid * seg), i1 = min(N, i0 + seg);
  int eq = 0;
  for (int i = i0; i < i1; ++i) eq += (valid(i) && key[i] == T) ? 1 : 0;
  int total;
  int rank = block_excl_scan(eq, sc, &total);
  for (int i = i0; i < i1; ++i) {
    if (!valid(i)) continue;
    const unsigned ki = key[i];
    if (ki > T) sel[i] = 1;
    else if (ki == T) { if (rank < r) sel[i] = 1; ++rank; }
  }
  __syncthreads();
}

// ascending list of the set positions of flag[0..N) -> out[]; returns the count.  Block-wide.
__device__ int block_compact(const unsigned char* flag, int N, int* out, Scratch* sc) {
  const int tid = threadIdx.x;
  const int seg = (N + kThreads - 1) / kThreads;
  const int i0 = min(N, tid * seg), i1 = min(N, i0 + seg);
  int cnt = 0;
  for (int i = i0; i < i1; ++i) cnt += flag[i] ? 1 : 0;
  int total;
  int pos = block_excl_scan(cnt, sc, &total);
  for (int i = i0; i < i1; ++i) if (flag[i]) out[pos++] = i;
  __syncthreads();
  return total;
}

// plain (coherent) streaming load: the pool is written by this kernel, so no .nc
__device__ __forceinline__ uint4 ld_stream16(const void* p) {
  uint4 r;
  asm volatile("ld.global.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_na16(void* p, const uint4& v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};"
               :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// a4: rows src_of(r) -> h + r for r in [0, moved), K and V together, in place, staged through REGISTERS.
// A chunk of rows_per_pass rows of K and of V is loaded completely (every thread holds its 16-byte vectors in
// registers: all loads of the chunk are in flight together), the block synchronises, then the chunk is written.
// src_of is increasing with src_of(r) >= h + r, so a chunk's writes never touch a row a later chunk still has
// to read.  Block-wide; s_off = [2][stage_rows] row offsets in shared memory.
template <typename SrcOf>
__device__ __forceinline__ void compact_rows_inplace(const Call& c, int layer, int s, int hk, int h, int moved, SrcOf src_of,
                                                     long long* s_off, int stage_rows) {
  const int tid = threadIdx.x;
  const int vpr = c.g.d / 8;                                   // 16-byte vectors per row
  constexpr int kVecPerThread = KARA_SEL_VEC;                  // per tensor
  const int rows_per_pass = kThreads * kVecPerThread / vpr;    // 128 rows at d = 128, 256 at d = 64
  __nv_bfloat16* kp = const_cast<__nv_bfloat16*>(c.k_pool);
  __nv_bfloat16* vp = const_cast<__nv_bfloat16*>(c.v_pool);
  for (int c0 = 0; c0 < moved; c0 += rows_per_pass) {
    const int rows = min(rows_per_pass, moved - c0);
    // the block-table walk once per row (the same for K and V), not once per 16-byte vector
    for (int r = tid; r < rows; r += kThreads) {
      const int row = c0 + r;
      s_off[r] = row_offset(c, layer, s, hk, src_of(row));
      s_off[stage_rows + r] = row_offset(c, layer, s, hk, h + row);
    }
    __syncthreads();
    uint4 kv[kVecPerThread], vv[kVecPerThread];
#pragma unroll
    for (int u = 0; u < kVecPerThread; ++u) {
      const int x = tid + u * kThreads;
      const int r = x / vpr, v = x % vpr;
      const long long off = r < rows ? s_off[r] : -1;
      kv[u] = off >= 0 ? __ldcg(reinterpret_cast<const uint4*>(kp + off + v * 8)) : make_uint4(0, 0, 0, 0);
      vv[u] = off >= 0 ? __ldcg(reinterpret_cast<const uint4*>(vp + off + v * 8)) : make_uint4(0, 0, 0, 0);
    }
    __syncthreads();                                           // every read of the chunk has completed
#pragma unroll
    for (int u = 0; u < kVecPerThread; ++u) {
      const int x = tid + u * kThreads;
      const int r = x / vpr, v = x % vpr;
      const long long off = r < rows ? s_off[stage_rows + r] : -1;
      if (off >= 0) { st_na16(kp + off + v * 8, kv[u]); st_na16(vp + off + v * 8, vv[u]); }
    }
    __syncthreads();
  }
}

__global__ void __launch_bounds__(kThreads, KARA_SEL_OCC) select_compact_kernel(const Call c, int stage_rows, int off_bytes) {
  // programmatic dependent launch: this grid may be scheduled while the score kernel drains; nothing the
  // score kernel writes is read before the wait, and the metadata kernel behind may be scheduled early too
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = c.n, n_pad = c.n_pad, k = c.k, keep = c.keep;
  // carve
  unsigned char* s_fill = smem_raw;                                            // [n_pad] fill flags
  float* s_A = reinterpret_cast<float*>(smem_raw + ((n_pad + 15) / 16) * 16);  // [n_pad]
  unsigned* s_key = reinterpret_cast<unsigned*>(s_A + n_pad);                  // [n_pad]
  int* s_I = reinterpret_cast<int*>(s_key + n_pad);                            // [k_pad]
  int* s_F = s_I + c.k_pad;                                                    // [keep_pad]
  unsigned* s_rkey = reinterpret_cast<unsigned*>(s_F + c.keep_pad);            // [k_pad] chunk keys
  Scratch* sc = reinterpret_cast<Scratch*>(s_rkey + c.k_pad);
  unsigned char* s_sel = reinterpret_cast<unsigned char*>(sc + 1);             // [n_pad] retained flag
  unsigned char* s_csel = s_sel + n_pad;                                       // [k_pad] chunk flags
  unsigned char* s_celig = s_csel + c.k_pad;                                   // [k_pad]
  long long* s_off = reinterpret_cast<long long*>(smem_raw + off_bytes);       // [2][stage_rows] src / dst offsets

  const int unit = blockIdx.x, tid = threadIdx.x;
  int li, s, w, hk;
  unit_decode(unit, c.n_seqs, c.n_windows, c.g.n_kv_heads, li, s, w, hk);
  const int layer = c.layer_begin + li;

  int h, t, len;                             // h = first window of the sequence, t = tail behind the last one
  if (!window_of(c, s, h, t, len)) return;   // uniform per CTA
  // every table entry of the window is validated BEFORE anything is written: a sequence with a block id
  // outside the pool is skipped as a whole (no compaction here, no metadata update in a5)
  if (!window_blocks_ok(c, s, h, len)) return;

  // ---- scores: sum the score kernel's partial column sums in part order -------------------
  const float* part = c.partial + (long long)unit * c.parts * n_pad;
  const int n_strips = strips_of_unit(unit, c.parts, c.part_T, c.part_nc, c.part_tpu);
  for (int j = tid; j < n_pad; j += kThreads) {
    float a = 0.f;
    if (j < n) for (int p = 0; p < n_strips; ++p) a += part[(long long)p * n_pad + j];
    s_A[j] = a;
    s_key[j] = key_of(a);
    s_sel[j] = 0;
    if (c.keep_debug && j < n) c.scores[(long long)unit * n_pad + j] = a;
  }
  for (int x = tid; x < c.k_pad; x += kThreads) { s_csel[x] = 0; s_celig[x] = 0; s_rkey[x] = 0u; }
  __syncthreads();

  // ---- a2: I = top-k (Eq. 5) ----------------------------------------------------------------
  block_top_m(s_key, n, k, [](int) { return true; }, s_sel, sc);
  block_compact(s_sel, n, s_I, sc);
  if (c.keep_debug) for (int x = tid; x < k; x += kThreads) c.idx_topk[(long long)unit * c.k_pad + x] = s_I[x];

  // ---- a3: Token2Chunk (Eq. 6-8) --------------------------------------------------------------
  int n_elig_local = 0;
  for (int x = tid; x < k - 1; x += kThreads) {
    const int a = s_I[x], b = s_I[x + 1];
    const int gap = b - a - 1;
    if (b - a < c.gamma && gap >= 1) {
      const float r = __fmul_rn(__fadd_rn(s_A[a], s_A[b]), (float)gap);   // Eq. 6, no contraction
      s_rkey[x] = key_of(r);
      s_celig[x] = 1;
      ++n_elig_local;
    }
  }
  int n_elig;
  block_excl_scan(n_elig_local, sc, &n_elig);
  __syncthreads();
  const int n_pick = min(c.P, n_elig);
  // top-P of the (few) eligible chunks under (R desc, ordinal asc) by direct ranking: a chunk is picked
  // iff fewer than n_pick eligible chunks precede it in that order
  for (int x = tid; x < k - 1; x += kThreads) {
    if (!s_celig[x]) continue;
    const unsigned rx = s_rkey[x];
    int before = 0;
    for (int y = 0; y < k - 1; ++y) {
      const unsigned ry = s_rkey[y];
      before += (s_celig[y] && (ry > rx || (ry == rx && y < x))) ? 1 : 0;
    }
    if (before < n_pick) s_csel[x] = 1;
  }
  __syncthreads();
  int added_local = 0;
  for (int x = tid; x < k - 1; x += kThreads)
    if (s_csel[x]) {
      for (int j = s_I[x] + 1; j < s_I[x + 1]; ++j) { s_sel[j] = 1; ++added_local; }   // Eq. 8
    }
  int added;
  block_excl_scan(added_local, sc, &added);
  __syncthreads();

  // ---- App. C.3 fill --------------------------------------------------------------------------
  {
    // Candidates are the positions unselected before the fill.  The histogram passes need a
    // stable candidate set, so the fill selects into its own flag array and the flags are merged
    // afterwards.
    const unsigned char* selc = s_sel;
    unsigned char* fillflag = s_fill;
    for (int j = tid; j < n; j += kThreads) fillflag[j] = 0;
    __syncthreads();
    block_top_m(s_key, n, keep - k - added, [selc](int j) { return selc[j] == 0; }, fillflag, sc);
    for (int j = tid; j < n; j += kThreads) if (fillflag[j]) s_sel[j] = 1;
    __syncthreads();
  }
  block_compact(s_sel, n, s_F, sc);   // F: ascending (reading G10), |F| = keep
  // F goes to the workspace for kara_gather_debug and, in a multi-window call, for compact_windows_kernel
  if (c.keep_debug || c.n_windows > 1)
    for (int x = tid; x < keep; x += kThreads) c.idx_final[(long long)unit * c.keep_pad + x] = s_F[x];
  if (c.n_windows > 1) return;               // a4 of a multi-window call: compact_windows_kernel

  // ---- a4: compaction of K and V (Eq. 9): rows h + F[c] -> h + c, buffer + tail rows behind them ----
  const int* F = s_F;
  compact_rows_inplace(c, layer, s, hk, h, keep + c.U + t,
                       [=](int row) { return row < keep ? h + F[row] : h + n + (row - keep); }, s_off, stage_rows);
}

// a4 of a multi-window call (App. C.2, reading G17): one CTA per (layer, sequence, KV head) moves, in window order,
//   new[h + w (keep+U) + c]        = old[h + w W + F_w[c]]       c < keep
//   new[h + w (keep+U) + keep + c] = old[h + w W + n + c]        c < U
//   new[h + NW (keep+U) + c]       = old[h + NW W + c]           c < t
// F_w is read from the workspace (written by select_compact_kernel of the same call).
__global__ void __launch_bounds__(kThreads, KARA_SEL_OCC) compact_windows_kernel(const Call c, int stage_rows) {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  long long* s_off = reinterpret_cast<long long*>(smem_raw);
  const int NW = c.n_windows, Hkv = c.g.n_kv_heads;
  const int hk = blockIdx.x % Hkv, s = (blockIdx.x / Hkv) % c.n_seqs, li = blockIdx.x / (Hkv * c.n_seqs);
  int h, t, len;
  if (!window_of(c, s, h, t, len)) return;
  if (!window_blocks_ok(c, s, h, len)) return;
  const int keep = c.keep, per = c.keep + c.U, n = c.n, W = c.W;
  const int32_t* F = c.idx_final + ((((long long)li * c.n_seqs + s) * NW) * Hkv + hk) * c.keep_pad;   // window 0
  const long long f_stride = (long long)Hkv * c.keep_pad;                                            // to the next window
  compact_rows_inplace(c, c.layer_begin + li, s, hk, h, NW * per + t,
                       [=](int row) {
                         if (row >= NW * per) return h + NW * W + (row - NW * per);       // tail
                         const int w = row / per, x = row - w * per;
                         return x < keep ? h + w * W + F[w * f_stride + x] : h + w * W + n + (x - keep);
                       }, s_off, stage_rows);
}

size_t smem_bytes(const Call& c) {
  size_t b = (size_t)((c.n_pad + 15) / 16) * 16;
  b += sizeof(float) * c.n_pad + sizeof(unsigned) * c.n_pad;
  b += sizeof(int) * (c.k_pad + c.keep_pad) + sizeof(unsigned) * c.k_pad;
  b += sizeof(Scratch);
  b += (size_t)c.n_pad + 2 * (size_t)c.k_pad;
  return (b + 15) / 16 * 16;   // the row-offset table [2][stage_rows] of int64 follows at this offset
}

}  // namespace

cudaError_t launch_select_compact(const Call& c, cudaStream_t st) {
  const int units = unit_count(c);
  // offset table: one pass of the compaction moves 256 x 8 vectors per tensor = at most 256 rows (d = 64)
  const int stage_rows = 256;
  const size_t off_bytes = smem_bytes(c);
  const size_t smem = off_bytes + 2 * sizeof(long long) * (size_t)stage_rows;
  cudaError_t e = cudaFuncSetAttribute(select_compact_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  // programmatic dependent launch behind the score kernel (see the kernel's first lines)
  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  cfg.gridDim = dim3(units); cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem; cfg.stream = st;
  return cudaLaunchKernelEx(&cfg, select_compact_kernel, c, stage_rows, (int)off_bytes);
}

cudaError_t launch_compact_windows(const Call& c, cudaStream_t st) {
  const int stage_rows = 256;
  const size_t smem = 2 * sizeof(long long) * (size_t)stage_rows;
  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  cfg.gridDim = dim3(c.n_layers * c.n_seqs * c.g.n_kv_heads); cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem; cfg.stream = st;
  return cudaLaunchKernelEx(&cfg, compact_windows_kernel, c, stage_rows);
}

}  // namespace kara
