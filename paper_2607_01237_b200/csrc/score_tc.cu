// score_tc.cu — a1 (Eq. 4): A = colsum(softmax(Q_W K_{W\\U}^T / sqrt(d))) on the
// 5th-generation tensor cores of sm_100a: TMA -> shared memory, tcgen05.mma -> TMEM, softmax out
// of TMEM, deterministic column sums.  DESIGN.md §Kernels/a1 has the derivation of every choice.
//
// Decomposition.  A unit is one (layer, sequence, KV head).  A query tile is 128 window tokens x
// ONE query head of the GQA group (rows of a row-softmax are independent, so any (token, head) ->
// row map is valid; TMA reads the rows at stride n_q_heads*d); with KARA_SCORE_QBUF_ONLY the U buffer
// tokens of several heads share a tile (box = tokens x heads, rows past the head group weigh 0).  All T = units * tiles_per_unit
// tiles of the launch form one sequence that is cut into n_clusters contiguous, equally long
// ranges (perfect balance; a range crosses unit boundaries, the part of a unit inside a range is
// a "segment").  A thread-block cluster of CL CTAs owns a range; CTA r of the cluster owns the
// 256 key rows [256 r, 256 r + 256) of the block-aligned key panel (whole paged blocks are
// loaded, one TMA box per block and 64-element column panel; rows outside the compressible
// region [h, h+n) are masked to -inf).  Per tile and CTA:
//   S[128 x 256] = Q_tile[128 x d] . K_cta[256 x d]^T      tcgen05.mma kind::f16, bf16 in, fp32 in TMEM,
//       issued as two N <= 128 halves, each with its own full / empty barrier, so a half is
//       refilled as soon as its column sums have been taken.
//   The softmax is split over SPECIALISED warps:
//   B warps (16: TMEM lane quadrant q x 32-column piece cq of each MMA half) — pass B, the only MUFU work.
//       One TMEM read, one write, in the 32x32b shape (four .x8 loads): a THREAD OWNS 32 CONSECUTIVE COLUMNS OF ONE ROW (a "piece",
//       one per half), so the maximum, the integer shift z = round(max c) (log2 domain) and the row sum
//       l = sum 2^(s c - z) are thread-local: no shuffle anywhere in the pass.  e = 2^(s c - z) is written
//       back in place; (z, l) per (row, 32-column piece) go to shared memory.
//   C warps (4: one per lane quadrant) — statistics, then pass C.  With lane = row, (z, l) of a row are merged
//       over its eight pieces and the CL CTAs with exact power-of-two rescaling built by integer arithmetic
//       (no MUFU); across CTAs with st.async + a transaction-count mbarrier per (buffer, quadrant) — no
//       fence, no cluster barrier.  The weight of (row, piece), w = 2^(z_piece - Z_row) / L_row, goes over
//       the piece's (z, l) entry as the pair {w, w}, ready for a packed FFMA2 (the four warps work on their
//       own quadrants in parallel: their shared-memory and MUFU.RCP operations queue behind the B warps'
//       exponentials, so the count of such operations per warp is what this step costs).  Pass C (one TMEM
//       read, 16x256b shape): acc_j += sum_i e_ij w_i in per-thread registers; with that load shape the
//       column sum over ALL tiles of a segment is a plain packed FFMA2; lanes are combined once per
//       segment.  Each TMEM half is handed back to the MMA warp as soon as it has been read.
// TMEM holds two 128 x 256 fp32 S buffers (all 512 columns).  The K panel is double-buffered so a
// segment change costs no bubble.
//
// Warp roles (768 threads): warps 0-15 B (q = warp & 3, piece cq = warp >> 2 of each MMA half), 16-19 C (q = warp & 3),
// 20 TMA producer, 21 MMA issuer, 22-23 idle (they complete the warpgroup whose registers setmaxnreg hands to
// the C warps).
// Output: partial[unit][p][j] (fp32), p = index of the range among those that touch the unit;
// the select kernel sums the strips in fixed order, so scores are bit-reproducible run to run
// (no atomics anywhere).
#include "score_tc_ptx.cuh"

namespace kara {

namespace {

constexpr int kBWarps = 16;                   // pass B warps: 0..15
constexpr int kCWarp0 = 16;                   // pass C warps: 16..19
constexpr int kProducerWarp = 20;
constexpr int kMmaWarp = 21;
constexpr int kThreads = 32 * 24;             // 6 warpgroups (setmaxnreg works per warpgroup)
// registers: 768 x 80 at launch; setmaxnreg only moves registers inside that allocation:
// 4 x 80 (B: two 32-register TMEM pieces in flight) + 120 (C: 64 accumulators + two 16-register pieces) + 40 (producer, MMA, idle) = 6 x 80
constexpr int kRegsB = 80, kRegsC = 120, kRegsOther = 40;
thread_local char g_tc_err[256] = "";


// ------------------------------------------------------------------------------------------------
// shared-memory carve-up (dynamic smem, manually aligned to 1024 B for the 128B swizzle)
// ------------------------------------------------------------------------------------------------
template <int D, int CL>
struct Smem {
  static constexpr int kPanels = D / 64;
  static constexpr int kKStages = CL >= 8 ? 1 : 2;   // 8-CTA clusters need the room for the exchange slots
  static constexpr int kQStages = 2;
  static constexpr int kKBytes = kPanels * kKeysPerCta * 128;
  static constexpr int kQStageBytes = kPanels * kTileM * 128;
  static constexpr int kOffK = 0;
  static constexpr int kOffQ = kOffK + kKStages * kKBytes;
  static constexpr int kOffColsum = kOffQ + kQStages * kQStageBytes;     // float [4 C warps][256]
  // per (buffer, piece column cq, row): {z, l} of the row's piece cq in half 0 and in half 1, written by the B warps,
  // overwritten by the C warps with the weight pairs {w0, w0, w1, w1}
  static constexpr int kOffRstat = kOffColsum + 4 * kKeysPerCta * 4;     // uint4 [2 bufs][4 cq][128 rows]
  static constexpr int kOffXch = kOffRstat + 2 * 4 * 128 * 16;           // uint2 [2 bufs][4 q][CL][32]
  static constexpr int kOffBars = kOffXch + 2 * 4 * CL * 32 * 8;
  // barriers: qfull[2] qempty[2] kfull[2] kempty[2] tfull[2][2] tempty[2][2] bdone[2] xbar[2][4] = 26 x 8 B
  static constexpr int kOffTmemPtr = kOffBars + 26 * 8;
  static constexpr int kBytes = kOffTmemPtr + 16;
  static constexpr int kAlloc = kBytes + 1024;   // slack for manual alignment
};

// One segment: the tiles [t0, t1) of `unit` that fall into this cluster's range.
struct Seg {
  int unit, part, li, s, w, hk, layer;
  int h, fb, off;          // window start, first key block (table index), h - fb*bs
  int c_lo, c_hi;          // this CTA's valid key columns [c_lo, c_hi) within its 256
  int n_cols;              // columns the MMAs of this CTA produce: valid columns rounded up to 16 (>= 16)
  int t0, t1;
  bool ok;
};

__device__ __forceinline__ Seg decode_seg(const Call& c, long long g, long long g_end, int rank, int cluster_id,
                                          int n_clusters, int T, int tpu) {
  Seg it;
  it.unit = (int)(g / tpu);
  it.t0 = (int)(g - (long long)it.unit * tpu);
  const long long left = g_end - g;
  it.t1 = (int)(left < (long long)(tpu - it.t0) ? it.t0 + left : tpu);
  it.part = cluster_id - tile_owner((long long)it.unit * tpu, n_clusters, T);
  unit_decode(it.unit, c.n_seqs, c.n_windows, c.g.n_kv_heads, it.li, it.s, it.w, it.hk);
  it.layer = c.layer_begin + it.li;
  const int len = c.seq_lens[it.s];
  const int h0 = c.win_start ? c.win_start[it.s] : len - c.n_windows * c.W;   // first window of the sequence
  const int t = len - h0 - c.n_windows * c.W;
  it.ok = (len >= 0 && h0 >= 0 && t >= 0 && ((len + c.g.bs - 1) >> c.g.bs_log2) <= c.max_blocks);
  it.h = it.ok ? h0 + it.w * c.W : 0;
  it.fb = it.h >> c.g.bs_log2;
  it.off = it.h - (it.fb << c.g.bs_log2);
  // panel row pr = rank*256 + col  <->  window-relative key j = pr - off ; valid iff 0 <= j < n
  const int lo = it.off - rank * kKeysPerCta, hi = it.off + c.n - rank * kKeysPerCta;
  it.c_lo = min(max(lo, 0), kKeysPerCta);
  it.c_hi = min(max(hi, 0), kKeysPerCta);
  if (!it.ok) it.c_lo = it.c_hi = 0;
  it.n_cols = max(16, (it.c_hi + 15) & ~15);
  return it;
}
// columns the MMA of half hf produces (0 = half not issued)
__device__ __forceinline__ int half_cols(int n_cols, int hf) { return min(max(n_cols - kHalf * hf, 0), kHalf); }

// ---- pass B on one piece: ONE row x 32 columns [col0, col0 + 32) of the CTA's 256 -------------------------
// x[i] = logit of column col0 + i; on return x[i] = e = 2^(s c - z) with the shift z = round(max c) of THIS
// piece (log2 domain), so e <= 2^0.5, and l = sum e.  Shifts are biased ints (the bit pattern of z + kMagic,
// see kZFloor); a fully masked piece has max = -inf -> as_int(t) < 0 -> z = floor, e = 0, l = 0.
template <bool RAGGED>
__device__ __forceinline__ void pass_b_body(uint32_t (&r)[32], int& z_out, float& l_out, float cs, int col0,
                                            int c_lo, int c_hi) {
  float x[32];
#pragma unroll
  for (int i = 0; i < 32; ++i) x[i] = __uint_as_float(r[i]);
  if (RAGGED) {
#pragma unroll
    for (int i = 0; i < 32; ++i)
      if (col0 + i < c_lo || col0 + i >= c_hi) x[i] = __int_as_float(0xff800000);
  }
  float m0 = max3(x[0], x[1], x[2]), m1 = max3(x[3], x[4], x[5]);
  float m2 = max3(x[6], x[7], x[8]), m3 = max3(x[9], x[10], x[11]);
  m0 = max3(m0, x[12], x[13]); m1 = max3(m1, x[14], x[15]);
  m2 = max3(m2, x[16], x[17]); m3 = max3(m3, x[18], x[19]);
  m0 = max3(m0, x[20], x[21]); m1 = max3(m1, x[22], x[23]);
  m2 = max3(m2, x[24], x[25]); m3 = max3(m3, x[26], x[27]);
  m0 = max3(m0, x[28], x[29]); m1 = max3(m1, x[30], x[31]);
  const float m = fmaxf(max3(m0, m1, m2), m3);
  // t = round(m c) + kMagic as a float; its bit pattern is the biased integer shift
  const float t = fminf(fmaf(m, cs, kMagic), kMagic + kZLim);
  const int z = max(kZFloor, __float_as_int(t));
  const float nz = kMagic - __int_as_float(z);                     // = -z, exact
  const uint64_t cs2 = pk2(cs, cs), nz2 = pk2(nz, nz);
  uint64_t la = pk2(0.f, 0.f), lb = pk2(0.f, 0.f);
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    float a, b;
    upk2(fma2(pk2(x[2 * i], x[2 * i + 1]), cs2, nz2), a, b);
    a = ex2(a); b = ex2(b);
    if (i & 1) lb = add2(lb, pk2(a, b)); else la = add2(la, pk2(a, b));
    r[2 * i] = __float_as_uint(a); r[2 * i + 1] = __float_as_uint(b);
  }
  float a, b;
  upk2(add2(la, lb), a, b);
  z_out = z;
  l_out = a + b;
}
// two copies of the body, so that the common (no ragged edge) path carries no select
// [colw, colw + colw_n) = the columns the WARP holds (the branch is warp-uniform), col0 = first of the thread's 32
__device__ __forceinline__ void pass_b_piece(uint32_t (&r)[32], int& z, float& l, float cs, int colw, int colw_n, int col0,
                                             int c_lo, int c_hi) {
  if (colw >= c_lo && colw + colw_n <= c_hi)    // false only on a ragged first / last chunk
    pass_b_body<false>(r, z, l, cs, col0, c_lo, c_hi);
  else
    pass_b_body<true>(r, z, l, cs, col0, c_lo, c_hi);
}

// ---- pass C on one loaded piece (16 rows x the 32 columns of piece PC): acc[PC*4 + i] (columns 32 PC + 8i+2qd+{0,1})
// += e(row) * w(row, piece).  r[4i+{0,1}] = row lr (+16 for the upper lanes), r[4i+{2,3}] = that row + 8; w0 / w1 = {w, w}
// of those two rows.
template <int PC>
__device__ __forceinline__ void pass_c_piece(const uint32_t (&r)[16], uint64_t (&acc)[32], uint64_t w0, uint64_t w1) {
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    uint64_t a = acc[PC * 4 + i];
    a = fma2(pk2u(r[4 * i], r[4 * i + 1]), w0, a);
    a = fma2(pk2u(r[4 * i + 2], r[4 * i + 3]), w1, a);
    acc[PC * 4 + i] = a;
  }
}

// ------------------------------------------------------------------------------------------------
// the kernel
// ------------------------------------------------------------------------------------------------
template <int D, int CL>
__global__ void __launch_bounds__(kThreads, 1)
score_tc_kernel(const __grid_constant__ CUtensorMap k_map, const __grid_constant__ CUtensorMap q_map,
                const Call c, int T, int tpu, int tok_tiles) {
  using SM = Smem<D, CL>;
  constexpr int QS = SM::kQStages;
  extern __shared__ unsigned char smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* gbase = smem_raw + (base - raw);
  const uint32_t sK = base + SM::kOffK;
  const uint32_t sQ = base + SM::kOffQ;
  float* colsum = reinterpret_cast<float*>(gbase + SM::kOffColsum);
  uint4* rstat = reinterpret_cast<uint4*>(gbase + SM::kOffRstat);
  uint2* xch = reinterpret_cast<uint2*>(gbase + SM::kOffXch);
  const uint32_t bars = base + SM::kOffBars;
  const uint32_t qfull = bars, qempty = bars + 16, kfull = bars + 32, kempty = bars + 48;
  const uint32_t tfull = bars + 64, tempty = bars + 96, bdone = bars + 128, xbar = bars + 144;
  volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(gbase + SM::kOffTmemPtr);

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;   // warp-uniform for the compiler
  const int rank = CL > 1 ? (int)cluster_ctarank() : 0;
  const int cluster_id = blockIdx.x / CL, n_clusters = gridDim.x / CL;
  const long long g_begin = (long long)cluster_id * T / n_clusters;
  const long long g_end = (long long)(cluster_id + 1) * T / n_clusters;

  if (threadIdx.x == 0) {
    for (int i = 0; i < 2; ++i) { mbar_init(qfull + 8 * i, 1); mbar_init(qempty + 8 * i, 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(kfull + 8 * i, 1); mbar_init(kempty + 8 * i, 1); }
    for (int i = 0; i < 4; ++i) {
      mbar_init(tfull + 8 * i, 1); mbar_init(tempty + 8 * i, 4);   // one arrive per C warp
    }
    for (int i = 0; i < 2; ++i) mbar_init(bdone + 8 * i, kBWarps);  // one arrive per B warp; all four C warps wait on it
    for (int i = 0; i < 8; ++i) mbar_init(xbar + 8 * i, 1);        // per (buffer, quadrant)
    fence_barrier_init();
  }
  if (warp == kMmaWarp) tmem_alloc(smem_u32((const void*)tmem_ptr), kTmemCols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (CL > 1) cluster_sync_all();
  const uint32_t tmem_base = *tmem_ptr;
  // programmatic dependent launch: the select/compaction grid may be scheduled as SMs drain (it waits for
  // this whole grid with griddepcontrol.wait before it reads anything)
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  if (warp >= kProducerWarp) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" :: "n"(kRegsOther));
  if (warp == kProducerWarp) {
    // ================================ TMA producer ==============================================
    const int blocks_per_cta = kKeysPerCta >> c.g.bs_log2;   // <= 16: one block per lane
    int q_iter = 0, k_iter = 0;
    long long g = g_begin;
    auto next_ok = [&](Seg& it) -> bool {
      while (g < g_end) {
        it = decode_seg(c, g, g_end, rank, cluster_id, n_clusters, T, tpu);
        g += it.t1 - it.t0;
        if (it.ok) return true;
      }
      return false;
    };
    // K panel of this CTA: whole blocks, skipped if they hold no compressible key
    auto load_k = [&](const Seg& it) {
      const int stage = k_iter % SM::kKStages, use = k_iter / SM::kKStages;
      ++k_iter;
      mbar_wait_backoff(kempty + 8 * stage, (use & 1) ^ 1);
      int my_bytes = 0, my_blk = -1, my_row = 0;
      if (lane < blocks_per_cta) {
        const int row0 = lane << c.g.bs_log2;                     // first panel row of this block in the CTA
        if (row0 < it.c_hi && row0 + c.g.bs > it.c_lo) {          // block intersects the valid columns
          const int tbl = it.fb + rank * blocks_per_cta + lane;
          if (tbl < c.max_blocks) {
            const int b = c.block_table[(long long)it.s * c.max_blocks + tbl];
            if (b >= 0 && b < c.g.num_blocks) { my_blk = b; my_row = row0; my_bytes = c.g.bs * D * 2; }
            else atomicOr(c.status, KARA_ST_BAD_BLOCK);
          }
        }
      }
      int tot = my_bytes;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
      if (lane == 0) mbar_expect_tx(kfull + 8 * stage, (uint32_t)tot);
      __syncwarp();
      if (my_blk >= 0) {
        const long long grow = (((long long)it.layer * c.g.num_blocks + my_blk) * c.g.n_kv_heads + it.hk) << c.g.bs_log2;
#pragma unroll
        for (int p = 0; p < SM::kPanels; ++p)
          tma_load_2d(sK + stage * SM::kKBytes + p * (kKeysPerCta * 128) + my_row * 128, &k_map, kfull + 8 * stage,
                      p * 64, (int)grow);
      }
      __syncwarp();
    };
    Seg cur, nxt;
    bool have = next_ok(cur);
    if (have) load_k(cur);
    while (have) {
      const bool have_n = next_ok(nxt);
      if (SM::kKStages == 2 && have_n) load_k(nxt);     // prefetch: its stage was released by the segment before `cur`
      if (lane == 0) {
        for (int tile = cur.t0; tile < cur.t1; ++tile, ++q_iter) {
          const int stage = q_iter % QS, use = q_iter / QS;
          mbar_wait_backoff(qempty + 8 * stage, (use & 1) ^ 1);
          mbar_expect_tx(qfull + 8 * stage, SM::kQStageBytes);
          // tile -> (head tile gq, token tile tt): rows = q_tile_toks tokens x 2^q_hpt_log2 heads (token-major in the box)
          const int gq = tile / tok_tiles, tt = tile % tok_tiles;
          const int tok = ((cur.li * c.n_seqs + cur.s) * c.n_windows + cur.w) * c.W + c.q_row_begin + tt * c.q_tile_toks;
#pragma unroll
          for (int p = 0; p < SM::kPanels; ++p)
            tma_load_3d(sQ + stage * SM::kQStageBytes + p * (kTileM * 128), &q_map, qfull + 8 * stage,
                        p * 64, cur.hk * c.G + (gq << c.q_hpt_log2), tok);
        }
      }
      __syncwarp();
      if (SM::kKStages == 1 && have_n) load_k(nxt);
      cur = nxt;
      have = have_n;
    }
  } else if (warp == kMmaWarp) {
    // ================================ MMA issuer ================================================
    // The whole warp walks the segments (warp-uniform values stay in uniform registers); one
    // elected lane issues.  Descriptor low words are base + compile-time offsets: shared-memory
    // addresses are < 2^18, so (addr >> 4) never carries out of the 14-bit address field.
    constexpr uint32_t kDescHi = (uint32_t)(1024u >> 4) | (1u << 14) | (2u << 29);   // SBO | version | SWIZZLE_128B
    constexpr uint32_t kDescLo = 1u << 16;                                           // LBO (unused)
    int q_iter = 0, k_iter = 0, tile_iter = 0;
    for (long long g = g_begin; g < g_end;) {
      int n_tiles, n_cols;
      {
        const Seg it = decode_seg(c, g, g_end, rank, cluster_id, n_clusters, T, tpu);
        n_tiles = it.t1 - it.t0;
        n_cols = it.ok ? it.n_cols : 0;
      }
      g += n_tiles;
      if (n_cols == 0) continue;
      const int kstage = k_iter % SM::kKStages, kuse = k_iter / SM::kKStages;
      ++k_iter;
      mbar_wait(kfull + 8 * kstage, kuse & 1);
      const uint32_t b_lo = ((sK + kstage * SM::kKBytes) >> 4) | kDescLo;
      for (int i = 0; i < n_tiles; ++i, ++q_iter, ++tile_iter) {
        const int stage = q_iter % QS, quse = q_iter / QS;
        const int buf = tile_iter & 1, tuse = tile_iter >> 1;
        mbar_wait(qfull + 8 * stage, quse & 1);
        const uint32_t a_lo = ((sQ + stage * SM::kQStageBytes) >> 4) | kDescLo;
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
          mbar_wait(tempty + 8 * (buf * 2 + hf), (tuse & 1) ^ 1);
          tc_fence_after();
          if (elect_one()) {
            const int nc = half_cols(n_cols, hf);
            if (nc > 0) {
              const uint32_t idesc = make_idesc_bf16(nc);
              const uint32_t d_tmem = tmem_base + buf * kKeysPerCta + hf * kHalf;
#pragma unroll
              for (int p = 0; p < SM::kPanels; ++p) {
#pragma unroll
                for (int ks = 0; ks < 4; ++ks) {
                  const uint64_t ad = ((uint64_t)kDescHi << 32) | (a_lo + ((p * (kTileM * 128) + ks * 32) >> 4));
                  const uint64_t bd = ((uint64_t)kDescHi << 32) |
                                      (b_lo + ((p * (kKeysPerCta * 128) + hf * (kHalf * 128) + ks * 32) >> 4));
                  umma_bf16(d_tmem, ad, bd, idesc, (p | ks) != 0);
                }
              }
            }
            umma_commit(tfull + 8 * (buf * 2 + hf));   // S half complete (fires at once if nothing was issued)
            if (hf == 1) {
              umma_commit(qempty + 8 * stage);         // Q stage reusable once these MMAs have read it
              if (i == n_tiles - 1) umma_commit(kempty + 8 * kstage);    // K stage reusable
            }
          }
          __syncwarp();
        }
      }
    }
  }
  } else if (warp >= kCWarp0) {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" :: "n"(kRegsC));
    // ================================ C warps: statistics + pass C ================================
    const int q = warp & 3;                              // TMEM lane quadrant
    const int qd = lane & 3, lr = lane >> 2;             // column pair within a group of 8; row within 8
    const uint32_t tq = tmem_base + ((uint32_t)(q * 32) << 16);
    uint64_t acc[32];
#pragma unroll
    for (int a = 0; a < 32; ++a) acc[a] = 0ull;
    int tile_iter = 0;
    for (long long g = g_begin; g < g_end;) {
      const Seg it = decode_seg(c, g, g_end, rank, cluster_id, n_clusters, T, tpu);
      g += it.t1 - it.t0;
      float* out = c.partial + ((long long)it.unit * c.parts + it.part) * c.n_pad;
      if (!it.ok) {
        // skipped unit: its strip must still be defined (zeros); the status word says why
        if (rank == 0) for (int j = threadIdx.x & 127; j < c.n_pad; j += 128) out[j] = 0.f;
        continue;
      }
      const int n_pieces = (it.n_cols + 31) >> 5;                       // 1 .. 8
      int tt = it.t0 % tok_tiles, gq = it.t0 / tok_tiles;               // token tile / head tile of `tile` (kept incrementally: no division per tile)
      for (int tile = it.t0; tile < it.t1; ++tile, ++tile_iter, gq += (tt + 1 == tok_tiles), tt = (tt + 1 == tok_tiles ? 0 : tt + 1)) {
        const int b = tile_iter & 1, par = (tile_iter >> 1) & 1;
        mbar_wait(bdone + 8 * b, par);                      // every B warp has written e back and left (z, l) per (row, piece)
        // the first TMEM read of pass C is requested now: it lands while the statistics below are merged
        tc_fence_after();
        const uint32_t ta = tq + b * kKeysPerCta, ta_hi = ta + (16u << 16);
        uint32_t ra[16], rb[16];
        tmem_ld_16x256b_x4(ta, ra);
        // ---- row statistics of this quadrant (lane = row): 8 pieces -> CTA -> cluster -> weights ----
        {
          uint4* ent = rstat + (size_t)(b * 4) * 128 + q * 32 + lane;
          int zp[8];                                         // zp[2 cq + hf]
          int z_row;
          float l_row = 0.f;
          {
            uint4 sc[4];
#pragma unroll
            for (int x = 0; x < 4; ++x) sc[x] = ent[x * 128];
#pragma unroll
            for (int x = 0; x < 4; ++x) { zp[2 * x] = (int)sc[x].x; zp[2 * x + 1] = (int)sc[x].z; }
            z_row = max(max(max(zp[0], zp[1]), max(zp[2], zp[3])), max(max(zp[4], zp[5]), max(zp[6], zp[7])));
#pragma unroll
            for (int x = 0; x < 4; ++x)
              l_row += __uint_as_float(sc[x].y) * pow2i(zp[2 * x] - z_row) + __uint_as_float(sc[x].w) * pow2i(zp[2 * x + 1] - z_row);
          }
          if (CL > 1) {
            // lane publishes its row to every peer CTA ...
            const uint32_t bar = xbar + 8 * (b * 4 + q);
            uint2* slot = xch + (size_t)(b * 4 + q) * CL * 32;
            if (lane == 0) mbar_expect_tx(bar, (CL - 1) * 32 * 8);
            __syncwarp();
            const uint32_t la = smem_u32(slot + rank * 32 + lane);
#pragma unroll
            for (int pr = 0; pr < CL; ++pr)
              if (pr != rank) st_async_b32x2(mapa(la, pr), (uint32_t)z_row, __float_as_uint(l_row), mapa(bar, pr));
            mbar_wait(bar, par);
            // ... and merges that row over the CTAs in rank order (identical bits on every CTA)
            int Z = z_row;
#pragma unroll
            for (int pr = 0; pr < CL; ++pr) if (pr != rank) Z = max(Z, (int)slot[pr * 32 + lane].x);
            float L = 0.f;
#pragma unroll
            for (int pr = 0; pr < CL; ++pr) {
              const uint2 v = slot[pr * 32 + lane];
              L += (pr == rank) ? l_row * pow2i(z_row - Z) : __uint_as_float(v.y) * pow2i((int)v.x - Z);
            }
            z_row = Z; l_row = L;
          }
          // tile row r = token r >> hpt_log2 of the tile, head r & (hpt - 1) of the head tile
          const int r = q * 32 + lane;
          const int tok = c.q_row_begin + tt * c.q_tile_toks + (r >> c.q_hpt_log2);
          const bool head_ok = (gq << c.q_hpt_log2) + (r & ((1 << c.q_hpt_log2) - 1)) < c.G;
          // 1 / L on the FMA pipe (a MUFU.RCP would queue behind the B warps' exponentials): the exponent-flip
          // estimate (12 % off at most) and three Newton steps, relative error < 1e-7
          float inv_row = __int_as_float(0x7EF311C7 - __float_as_int(l_row));
#pragma unroll
          for (int nr = 0; nr < 3; ++nr) inv_row = inv_row * fmaf(-l_row, inv_row, 2.f);
          if (!(l_row > 0.f) || tok >= c.W || !head_ok) inv_row = 0.f;   // rows past the window / the head group contribute nothing
          // the weights of (row, piece cq of half 0 / half 1) go over the entry as the pairs {w0, w0, w1, w1}
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const uint32_t w0 = __float_as_uint(inv_row * pow2i(zp[2 * x] - z_row));
            const uint32_t w1 = __float_as_uint(inv_row * pow2i(zp[2 * x + 1] - z_row));
            ent[x * 128] = make_uint4(w0, w0, w1, w1);
          }
          __syncwarp();
        }
        tc_fence_after();
        // weights: rows lr + 8k (k = 0..3) x pieces 0..7, {w, w} pairs, fetched just before their use
        const uint2* wrow = reinterpret_cast<const uint2*>(rstat + (size_t)(b * 4) * 128 + q * 32 + lr);
        auto wld = [&](int pc, int k) -> uint64_t {        // piece pc = 4 hf + cq in column order
          const uint2 v = wrow[(size_t)((pc & 3) * 128 + 8 * k) * 2 + (pc >> 2)];
          return pk2u(v.x, v.y);
        };
        // ---- pass C: acc_j += sum_i e_ij w_i, piece by piece (16 rows x 32 columns per TMEM read, the next read in flight
        // under the FFMA2s of the current one); each half is handed back to the MMA warp as soon as it has been read ----
#define KARA_C_STEP(PC)                                                                   \
        if (PC < n_pieces) {                                                              \
          const uint64_t w0 = wld(PC, 0), w1 = wld(PC, 1), v0 = wld(PC, 2), v1 = wld(PC, 3); \
          tmem_wait_ld();                                                                 \
          tmem_ld_16x256b_x4(ta_hi + 32 * PC, rb);                                        \
          pass_c_piece<PC>(ra, acc, w0, w1);                                              \
          tmem_wait_ld();                                                                 \
          if (PC + 1 < n_pieces) tmem_ld_16x256b_x4(ta + 32 * (PC + 1), ra);              \
          pass_c_piece<PC>(rb, acc, v0, v1);                                              \
        }
        KARA_C_STEP(0) KARA_C_STEP(1) KARA_C_STEP(2) KARA_C_STEP(3)
        // half 0 has been read completely: the MMA may refill it
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty + 8 * (b * 2 + 0));
        KARA_C_STEP(4) KARA_C_STEP(5) KARA_C_STEP(6) KARA_C_STEP(7)
#undef KARA_C_STEP
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty + 8 * (b * 2 + 1));
      }

      // ---- segment done: combine lanes (fixed order), then the 4 warps (fixed order), write the strip ----
#pragma unroll
      for (int a = 0; a < 32; ++a) {
        float v0, v1;
        upk2(acc[a], v0, v1);
        v0 += __shfl_xor_sync(0xffffffffu, v0, 4);  v1 += __shfl_xor_sync(0xffffffffu, v1, 4);
        v0 += __shfl_xor_sync(0xffffffffu, v0, 8);  v1 += __shfl_xor_sync(0xffffffffu, v1, 8);
        v0 += __shfl_xor_sync(0xffffffffu, v0, 16); v1 += __shfl_xor_sync(0xffffffffu, v1, 16);
        if (lr == 0)
          *reinterpret_cast<float2*>(&colsum[q * kKeysPerCta + (a >> 3) * 64 + (a & 7) * 8 + 2 * qd]) = make_float2(v0, v1);
        acc[a] = 0ull;
      }
      named_bar_sync(1, 128);
#pragma unroll
      for (int xx = 0; xx < 2; ++xx) {
        const int x = (threadIdx.x & 127) + 128 * xx;
        float v = 0.f;
#pragma unroll
        for (int wv = 0; wv < 4; ++wv) v += colsum[wv * kKeysPerCta + x];
        if (x >= it.c_lo && x < it.c_hi) out[rank * kKeysPerCta + x - it.off] = v;
      }
      named_bar_sync(1, 128);
    }
  } else {
    // ================================ B warps: pass B ================================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" :: "n"(kRegsB));
    // Every thread owns, in EACH MMA half, one piece: 32 consecutive columns [32 pcq, + 32) of the half, of one S row.
    // All 16 warps sweep half 0, then half 1, so the refill of a half has a whole half-sweep of slack and four warps per
    // scheduler feed the MUFU pipe at any time.
    const int q = warp & 3, cq = warp >> 2;
    // 32x32b: warp (q, cq) holds rows [32 q, + 32) x piece column cq; thread = TMEM lane
    const int pcq = cq, colw0 = cq * 32, colw_n = 32;
    const int row = q * 32 + lane;
    const uint32_t tq = tmem_base + ((uint32_t)(q * 32) << 16) + cq * 32;
    const float cs = kLog2e * rsqrtf((float)D);
    int tile_iter = 0;
    for (long long g = g_begin; g < g_end;) {
      const Seg it = decode_seg(c, g, g_end, rank, cluster_id, n_clusters, T, tpu);
      g += it.t1 - it.t0;
      if (!it.ok) continue;
      const int c_lo = it.c_lo, c_hi = it.c_hi;
      // the MMA writes (some of) this warp's 64 columns of half 0 / 1 (a piece beyond them is masked as a whole)
      const bool act0 = colw0 < it.n_cols, act1 = kHalf + colw0 < it.n_cols;
      for (int tile = it.t0; tile < it.t1; ++tile, ++tile_iter) {
        const int b = tile_iter & 1, par = (tile_iter >> 1) & 1;
        const uint32_t ta = tq + b * kKeysPerCta;
        int z0 = kZFloor, z1 = kZFloor;
        float l0 = 0.f, l1 = 0.f;
        uint32_t ra[32], rb[32];
        mbar_wait(tfull + 8 * (b * 2 + 0), par);
        tc_fence_after();
        tmem_ld_32x32b_x32(ta, ra);                      // (an inactive piece is loaded too and ignored)
        // the TMEM load of piece 1 runs under the exponentials of piece 0 (in the B-bound steady state its S half
        // has landed long before; a starved B warp loses at most the time between the two MMA halves here)
        tmem_wait_ld();
        // ---- pass B: e = 2^(s c - z) in place; (z, l) of (row, piece); the thread owns row 32 q + lane ----
        if (act0) {
          pass_b_piece(ra, z0, l0, cs, colw0, colw_n, pcq * 32, c_lo, c_hi);
          tmem_st_32x32b_x32(ta, ra);
        }
        mbar_wait(tfull + 8 * (b * 2 + 1), par);
        tc_fence_after();
        tmem_ld_32x32b_x32(ta + kHalf, rb);
        tmem_wait_ld();
        if (act1) {
          pass_b_piece(rb, z1, l1, cs, kHalf + colw0, colw_n, kHalf + pcq * 32, c_lo, c_hi);
          tmem_st_32x32b_x32(ta + kHalf, rb);
        }
        rstat[(b * 4 + pcq) * 128 + row] = make_uint4((uint32_t)z0, __float_as_uint(l0), (uint32_t)z1, __float_as_uint(l1));
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bdone + 8 * b);
      }
    }
  }

  // ---- teardown: nobody may exit while a peer can still write into this CTA ----
  tc_fence_before();
  __syncthreads();
  if (CL > 1) cluster_sync_all();
  if (warp == kMmaWarp) { tc_fence_after(); tmem_dealloc(tmem_base, kTmemCols); }
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

int tc_fail(int code, const char* msg) {
  snprintf(g_tc_err, sizeof g_tc_err, "%s", msg);
  return code;
}

int cluster_size_for(const Call& c) {
  const int rows = c.n + c.g.bs - 1;                 // worst-case alignment of the window start
  const int need = (rows + kKeysPerCta - 1) / kKeysPerCta;
  return need <= 1 ? 1 : need <= 2 ? 2 : need <= 4 ? 4 : need <= 8 ? 8 : 0;
}

template <int D, int CL>
int launch_impl(ScoreTcState* s, Call& c, cudaStream_t st) {
  using SM = Smem<D, CL>;
  auto kern = score_tc_kernel<D, CL>;
  // per launch: the attribute belongs to the current device / context, not to the process
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SM::kAlloc) != cudaSuccess)
    return tc_fail(KARA_ECUDA, "cudaFuncSetAttribute(max dynamic smem) failed");
  const int tok_tiles = (c.W - c.q_row_begin + c.q_tile_toks - 1) / c.q_tile_toks;
  const int hpt = 1 << c.q_hpt_log2;
  const int tpu = tok_tiles * ((c.G + hpt - 1) / hpt);
  const int units = unit_count(c);
  const long long T = (long long)units * tpu;
  if (T >= (1ll << 31)) return tc_fail(KARA_EUNSUPPORTED, "more than 2^31 query tiles in one call");

  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = CL; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = SM::kAlloc;
  cfg.stream = st;
  int max_clusters = 0;
  cfg.gridDim = dim3(CL * (s->num_sms / CL));
  if (cudaOccupancyMaxActiveClusters(&max_clusters, kern, &cfg) != cudaSuccess || max_clusters <= 0) {
    cudaGetLastError();
    max_clusters = s->num_sms / CL;
  }
  if (max_clusters > kMaxSms) max_clusters = kMaxSms;
  const int n_clusters = (int)(T < max_clusters ? T : max_clusters);
  cfg.gridDim = dim3(CL * n_clusters);
  c.part_T = (int)T; c.part_nc = n_clusters; c.part_tpu = tpu;
  // every unit's strips must fit the workspace stride (strips_bound is the proof; this is the check)
  const long long per_range = T / n_clusters;
  long long ranges = (tpu - 1 + per_range - 1) / per_range + 1;
  if (ranges > tpu) ranges = tpu;
  if (kScoreStrips * ranges > c.parts) return tc_fail(KARA_ENOMEM, "workspace holds too few partial-score strips per unit");

  CUtensorMap kmap, qmap;
  memcpy(&kmap, s->k_map, sizeof kmap);
  memcpy(&qmap, s->q_map, sizeof qmap);
  cudaError_t e = cudaLaunchKernelEx(&cfg, kern, kmap, qmap, (const Call)c, (int)T, tpu, tok_tiles);
  if (e != cudaSuccess) return tc_fail(KARA_ECUDA, cudaGetErrorString(e));
  return KARA_OK;
}

}  // namespace

const char* score_tc_error() { return g_tc_err; }


int score_tc_attach(ScoreTcState* s, const Geom& g, void* k_pool) {
  s->ready = false;
  s->q_ptr = nullptr;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return KARA_OK; }   // no device: SIMT path errors later
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { cudaGetLastError(); return KARA_OK; }
  s->num_sms = prop.multiProcessorCount;
  if (prop.major != 10) return KARA_OK;                // not a tcgen05 part: SIMT kernel only
  EncodeTiledFn enc = get_encode();
  if (!enc) return tc_fail(KARA_ECUDA, "cuTensorMapEncodeTiled entry point not found");
  const unsigned long long rows = (unsigned long long)g.n_layers * g.num_blocks * g.n_kv_heads * g.bs;
  if (rows >= (1ull << 31)) return KARA_OK;            // beyond one tensor map's signed coordinates: SIMT path
  cuuint64_t dims[2] = {(cuuint64_t)g.d, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)g.d * 2};
  cuuint32_t box[2] = {64u, (cuuint32_t)g.bs};
  cuuint32_t estr[2] = {1u, 1u};
  CUtensorMap m;
  CUresult r = enc(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, k_pool, dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    snprintf(g_tc_err, sizeof g_tc_err, "cuTensorMapEncodeTiled(K pool) failed: CUresult %d", (int)r);
    return KARA_ECUDA;
  }
  memcpy(s->k_map, &m, sizeof m);
  s->ready = true;
  return KARA_OK;
}

const char* score_tc_unsupported_reason(const ScoreTcState& s, const Call& c) {
  if (!s.ready) return "no sm_100 device, or the K pool has 2^31 rows or more (beyond one tensor map's coordinates)";
  if (c.g.d != 64 && c.g.d != 128) return "head_dim not 64 or 128";
  if (c.g.bs > kKeysPerCta) return "block_size above 256";
  if (cluster_size_for(c) == 0) return "window needs more than 8 CTAs of 256 keys";
  const unsigned long long toks = (unsigned long long)c.n_layers * c.n_seqs * c.n_windows * c.W;
  if (toks >= (1ull << 31)) return "2^31 window tokens or more in one call";
  return nullptr;
}
bool score_tc_supported(const ScoreTcState& s, const Call& c) { return score_tc_unsupported_reason(s, c) == nullptr; }

int score_tc_launch(ScoreTcState* s, Call& c, cudaStream_t st, int* n_launches) {
  // window_q tensor map: [d][n_q_heads][layers*seqs*W tokens], box 64 x heads-per-tile x tokens-per-tile (= 128 rows), 128B swizzle
  const long long key[6] = {(long long)(uintptr_t)c.window_q, c.g.d, c.n_q_heads, (long long)c.n_layers * c.n_seqs * c.n_windows * c.W, c.q_tile_toks, c.q_hpt_log2};
  if (s->q_ptr != c.window_q || memcmp(key, s->q_key, sizeof key) != 0) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return tc_fail(KARA_ECUDA, "cuTensorMapEncodeTiled entry point not found");
    cuuint64_t dims[3] = {(cuuint64_t)c.g.d, (cuuint64_t)c.n_q_heads, (cuuint64_t)key[3]};
    cuuint64_t strides[2] = {(cuuint64_t)c.g.d * 2, (cuuint64_t)c.g.d * 2 * c.n_q_heads};
    cuuint32_t box[3] = {64u, (cuuint32_t)(1 << c.q_hpt_log2), (cuuint32_t)c.q_tile_toks};   // 128 rows: tokens x heads
    cuuint32_t estr[3] = {1u, 1u, 1u};
    CUtensorMap m;
    CUresult r = enc(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<__nv_bfloat16*>(c.window_q), dims, strides,
                     box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
      snprintf(g_tc_err, sizeof g_tc_err, "cuTensorMapEncodeTiled(window_q) failed: CUresult %d", (int)r);
      return KARA_ECUDA;
    }
    memcpy(s->q_map, &m, sizeof m);
    s->q_ptr = c.window_q;
    memcpy(s->q_key, key, sizeof key);
  }
  const int cl = cluster_size_for(c);
  int rc = KARA_EUNSUPPORTED;
#define KARA_DISPATCH(DD, CC) if (c.g.d == DD && cl == CC) rc = launch_impl<DD, CC>(s, c, st);
  KARA_DISPATCH(64, 1) KARA_DISPATCH(64, 2) KARA_DISPATCH(64, 4) KARA_DISPATCH(64, 8)
  KARA_DISPATCH(128, 1) KARA_DISPATCH(128, 2) KARA_DISPATCH(128, 4) KARA_DISPATCH(128, 8)
#undef KARA_DISPATCH
  if (rc == KARA_OK && n_launches) *n_launches = 1;
  return rc;
}

}  // namespace kara

