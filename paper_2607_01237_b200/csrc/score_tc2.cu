// score_tc2.cu — a1 (Eq. 4), TWO-PHASE variant of the tcgen05 score kernel (KARA_SCORE_TWO_PHASE).
//
// Same decomposition as score_tc.cu (units, 128-row query tiles of one query head, one contiguous range of
// tiles per cluster, CTA r owns key rows [256 r, 256 r + 256) of the block-aligned key panel), same TMA /
// tcgen05 plumbing, same statistics conventions.  What differs is how the two passes over S are made.
// score_tc.cu writes e = 2^(s c - z) back to TMEM and reads it again for the normalised column sums, which
// ties pass B, the statistics, pass C and the refill of the TMEM buffer into one latency ring.  Here S is
// COMPUTED TWICE instead (the tensor pipe is a quarter busy):
//   phase 1  MMA1 -> TMEM region A.  8 warps read S once and keep only the row statistics (z, l); all
//            exponentials of this phase run on the FMA pipe (degree-3 exp2, error 7.5e-5, which scales a
//            whole row); nothing is written back, the region is released as soon as the loads have landed.
//   S warps  (z, l) of a row over the two halves and the CL CTAs (st.async exchange), then
//            o = Z + log2 L per row to shared memory.
//   phase 2  one tile behind: MMA2 -> TMEM region B recomputes S; 8 warps read it once and add
//            2^(s c - o) — the softmax probability itself, one MUFU ex2 per element — straight into the
//            per-thread column sums.  No TMEM store, no second read, no dependency of the refill on phase 2's
//            arithmetic.
// Q tiles live in a 3-stage ring (a tile serves MMA1 and, one step later, MMA2); one K panel per segment.
// Measured (round 1, cfg2): correct (score error 0.7 % of the tolerance) but 309 us against 200 us of
// score_tc.cu: phase 1 costs 8 FMA-lane operations per element, i.e. 2,048 cycles per tile on the FMA pipe —
// as much as phase 2 on the MUFU pipe — and about 1,000 issued instructions per tile and warp.  Kept
// selectable as the base of the next round's work (DESIGN.md §10 has the measurements).
//
// Warp roles (768 threads): warps 0-7 phase 1 (q = warp & 3, hf = warp >> 2), 8-15 phase 2 (same map),
// 16-19 statistics (q = warp & 3), 20 TMA producer, 21 MMA issuer, 22-23 idle.
// Output: partial[unit][p][j] (fp32) as in score_tc.cu; bit-reproducible run to run (no atomics).
#include "score_tc_ptx.cuh"

namespace kara {

namespace {

constexpr int kP2Warp0 = 8;                   // phase-1 warps: 0..7, phase-2 warps: 8..15
constexpr int kSWarp0 = 16;                   // statistics warps: 16..19
constexpr int kProducerWarp = 20;
constexpr int kMmaWarp = 21;
constexpr int kThreads = 32 * 24;             // 6 warpgroups (setmaxnreg works per warpgroup); warps 22, 23 idle
// registers: 768 x 80 at launch; setmaxnreg only moves registers inside that allocation:
// 2 x 88 (phase 1) + 2 x 112 (phase 2) + 40 (S) + 40 (producer, MMA, idle) <= 6 x 80
constexpr int kRegsP1 = 88, kRegsP2 = 112, kRegsOther = 40;
constexpr int kSlots = 4;                     // statistics slots between phase 1, the S warps and phase 2
#ifndef KARA_P1_MUFU_MASK
#define KARA_P1_MUFU_MASK 0x22                // groups 1 and 5 of 8: a quarter of phase 1's exponentials on the MUFU pipe
#endif
constexpr unsigned kP1MufuMask = KARA_P1_MUFU_MASK;
char g_tc_err[256] = "";

// ------------------------------------------------------------------------------------------------
// shared-memory carve-up (dynamic smem, manually aligned to 1024 B for the 128B swizzle)
// ------------------------------------------------------------------------------------------------
template <int D, int CL>
struct Smem {
  static constexpr int kPanels = D / 64;
  static constexpr int kKStages = 1;                 // (the producer code is written for 1 or 2)
  static constexpr int kQStages = 3;                 // Q(t) serves MMA1(t) and, one step later, MMA2(t)
  static constexpr int kKBytes = kPanels * kKeysPerCta * 128;
  static constexpr int kQStageBytes = kPanels * kTileM * 128;
  static constexpr int kOffK = 0;                    // one K panel (both phases of a segment read it)
  static constexpr int kOffQ = kOffK + kKBytes;
  static constexpr int kOffColsum = kOffQ + kQStages * kQStageBytes;     // float [4 quadrants][256]
  // statistics slots: phase 1 may run up to kQStages - 1 = 2 tiles ahead of phase 2, so everything that is
  // handed from phase 1 over the S warps to phase 2 lives in kSlots = 4 slots (tile & 3)
  static constexpr int kOffOrow = kOffColsum + 4 * kKeysPerCta * 4;      // float [4 slots][4 q][32 rows]: Z + log2 L of the row
  static constexpr int kOffRstat = kOffOrow + kSlots * 4 * 32 * 4;       // uint2 [4 slots][2 halves][128 rows]
  static constexpr int kOffXch = kOffRstat + kSlots * 2 * 128 * 8;       // uint2 [4 slots][4 q][CL][32]
  static constexpr int kOffBars = kOffXch + kSlots * 4 * CL * 32 * 8;
  // barriers: qfull[3] qempty[3] kfull kempty tfull1[2] tempty1[2] tfull2[2] tempty2[2] bdone1[4] xbar[4][4] zready[4][4] = 52 x 8 B
  static constexpr int kOffTmemPtr = kOffBars + 52 * 8;
  static constexpr int kBytes = kOffTmemPtr + 16;
  static constexpr int kAlloc = kBytes + 1024;   // slack for manual alignment
};

// One segment: the tiles [t0, t1) of `unit` that fall into this cluster's range.
struct Seg {
  int unit, part, li, s, hk, layer;
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
  unit_decode(it.unit, c.n_seqs, c.g.n_kv_heads, it.li, it.s, it.hk);
  it.layer = c.layer_begin + it.li;
  const int len = c.seq_lens[it.s];
  it.h = c.win_start ? c.win_start[it.s] : len - c.W;
  const int t = len - it.h - c.W;
  it.ok = (it.h >= 0 && t >= 0 && ((len + c.g.bs - 1) >> c.g.bs_log2) <= c.max_blocks);
  if (!it.ok) it.h = 0;
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

// ---- phase 1 on one piece: 2 rows (K0, K0+1) x 16 columns of a 64-column chunk --------------------------
// r[4i+j] = row K0, r[4i+2+j] = row K0+1, column col0 + 8 i + 2 qd + j of the CTA's 256.  Only the row
// statistics are wanted: running (z, l) per row with exact power-of-two rescaling — the shift of the piece
// is z = max(z_run, round(m c)), an integer in the log2 domain carried as a biased int (see kZFloor), so
// e <= 2^0.5 and l_run is rescaled by 2^(z_old - z) built from the exponent field.  All exponentials of this
// phase run on the FMA pipe (exp2_poly2): the MUFU pipe belongs to phase 2.  A masked column has
// x = -inf -> clamped to 2^-125, which vanishes in l.
template <int K0, bool RAGGED>
__device__ __forceinline__ void stats_body(const uint32_t (&rin)[32], int (&zrun)[4], float (&lrun)[4], float cs,
                                           int qd, int col0, int c_lo, int c_hi) {
  float x[32];
#pragma unroll
  for (int i = 0; i < 32; ++i) x[i] = __uint_as_float(rin[i]);
  if (RAGGED) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int col = col0 + 8 * i + 2 * qd + j;
        if (col < c_lo || col >= c_hi) { x[4 * i + j] = __int_as_float(0xff800000); x[4 * i + 2 + j] = __int_as_float(0xff800000); }
      }
    }
  }
  float m0 = max3(x[0], x[1], x[4]), m1 = max3(x[2], x[3], x[6]);
  float m0b = max3(x[5], x[8], x[9]), m1b = max3(x[7], x[10], x[11]);
  m0 = max3(m0, x[12], x[13]);   m1 = max3(m1, x[14], x[15]);
  m0b = max3(m0b, x[16], x[17]); m1b = max3(m1b, x[18], x[19]);
  m0 = max3(m0, x[20], x[21]);   m1 = max3(m1, x[22], x[23]);
  m0b = max3(m0b, x[24], x[25]); m1b = max3(m1b, x[26], x[27]);
  m0 = max3(m0, x[28], x[29]);   m1 = max3(m1, x[30], x[31]);
  m0 = fmaxf(m0, m0b);           m1 = fmaxf(m1, m1b);
  // t = round(m c) + kMagic as a float; its bit pattern is the biased integer shift
  const float t0 = fminf(fmaf(m0, cs, kMagic), kMagic + kZLim);
  const float t1 = fminf(fmaf(m1, cs, kMagic), kMagic + kZLim);
  // (a tile starts at (z, l) = (floor, 0), for which this update is exact: one code path for every chunk)
  const int z0 = max(zrun[K0], __float_as_int(t0)), z1 = max(zrun[K0 + 1], __float_as_int(t1));
  const float l0s = lrun[K0] * pow2i(zrun[K0] - z0), l1s = lrun[K0 + 1] * pow2i(zrun[K0 + 1] - z1);
  zrun[K0] = z0; zrun[K0 + 1] = z1;
  const float nz0 = kMagic - __int_as_float(z0), nz1 = kMagic - __int_as_float(z1);   // = -z, exact
  const uint64_t cs2 = pk2(cs, cs), nz0_2 = pk2(nz0, nz0), nz1_2 = pk2(nz1, nz1);
  uint64_t l0 = pk2(l0s, 0.f), l1 = pk2(l1s, 0.f);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    // kP1MufuMask: column groups of phase 1 that use the MUFU pipe's spare share instead of the polynomial
    float a, b;
    if ((kP1MufuMask >> i) & 1) { upk2(fma2(pk2(x[4 * i], x[4 * i + 1]), cs2, nz0_2), a, b); a = ex2(a); b = ex2(b); }
    else exp2_poly2(fma2(pk2(x[4 * i], x[4 * i + 1]), cs2, nz0_2), a, b);
    l0 = add2(l0, pk2(a, b));
    if ((kP1MufuMask >> i) & 1) { upk2(fma2(pk2(x[4 * i + 2], x[4 * i + 3]), cs2, nz1_2), a, b); a = ex2(a); b = ex2(b); }
    else exp2_poly2(fma2(pk2(x[4 * i + 2], x[4 * i + 3]), cs2, nz1_2), a, b);
    l1 = add2(l1, pk2(a, b));
  }
  float a, b;
  upk2(l0, a, b); lrun[K0] = a + b;
  upk2(l1, a, b); lrun[K0 + 1] = a + b;
}
// two copies of the body, so that the common (no ragged edge) path carries no selects
template <int K0>
__device__ __forceinline__ void stats_piece(const uint32_t (&rin)[32], int (&zrun)[4], float (&lrun)[4], float cs,
                                            int qd, int col0, int c_lo, int c_hi) {
  if (col0 >= c_lo && col0 + 64 <= c_hi)        // warp-uniform: false only on the ragged first / last chunk
    stats_body<K0, false>(rin, zrun, lrun, cs, qd, col0, c_lo, c_hi);
  else
    stats_body<K0, true>(rin, zrun, lrun, cs, qd, col0, c_lo, c_hi);
}

// ---- phase 2 on one piece: acc[i] (columns 8i+2qd+{0,1} of the chunk) += 2^(s c - o_row) for its 2 rows;
//      o_row = Z + log2 L of the row (phase 1), so the terms are the softmax probabilities themselves ----
__device__ __forceinline__ void score_piece(const uint32_t (&r)[32], uint64_t (&acc)[8], float cs, float oa, float ob) {
  const uint64_t cs2 = pk2(cs, cs), na = pk2(-oa, -oa), nb = pk2(-ob, -ob);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    float a0, a1, b0, b1;
    upk2(fma2(pk2u(r[4 * i], r[4 * i + 1]), cs2, na), a0, a1);
    upk2(fma2(pk2u(r[4 * i + 2], r[4 * i + 3]), cs2, nb), b0, b1);
    a0 = ex2(a0); a1 = ex2(a1); b0 = ex2(b0); b1 = ex2(b1);
    acc[i] = add2(add2(acc[i], pk2(a0, a1)), pk2(b0, b1));
  }
}

// ------------------------------------------------------------------------------------------------
// the kernel
// ------------------------------------------------------------------------------------------------
template <int D, int CL>
__global__ void __launch_bounds__(kThreads, 1)
score_tc2_kernel(const __grid_constant__ CUtensorMap k_map, const __grid_constant__ CUtensorMap q_map,
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
  float* orow = reinterpret_cast<float*>(gbase + SM::kOffOrow);
  uint2* rstat = reinterpret_cast<uint2*>(gbase + SM::kOffRstat);
  uint2* xch = reinterpret_cast<uint2*>(gbase + SM::kOffXch);
  const uint32_t bars = base + SM::kOffBars;
  const uint32_t qfull = bars, qempty = bars + 24, kfull = bars + 48, kempty = bars + 56;
  const uint32_t tfull1 = bars + 64, tempty1 = bars + 80, tfull2 = bars + 96, tempty2 = bars + 112;
  const uint32_t bdone1 = bars + 128, xbar = bars + 160, zready = bars + 288;
  volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(gbase + SM::kOffTmemPtr);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rank = CL > 1 ? (int)cluster_ctarank() : 0;
  const int cluster_id = blockIdx.x / CL, n_clusters = gridDim.x / CL;
  const long long g_begin = (long long)cluster_id * T / n_clusters;
  const long long g_end = (long long)(cluster_id + 1) * T / n_clusters;

  if (threadIdx.x == 0) {
    for (int i = 0; i < 3; ++i) { mbar_init(qfull + 8 * i, 1); mbar_init(qempty + 8 * i, 1); }
    mbar_init(kfull, 1); mbar_init(kempty, 1);
    for (int i = 0; i < 2; ++i) {
      mbar_init(tfull1 + 8 * i, 1); mbar_init(tempty1 + 8 * i, 4);   // one arrive per phase-1 warp of the half
      mbar_init(tfull2 + 8 * i, 1); mbar_init(tempty2 + 8 * i, 4);   // one arrive per phase-2 warp of the half
    }
    for (int i = 0; i < kSlots; ++i) mbar_init(bdone1 + 8 * i, 8);   // one arrive per phase-1 warp
    for (int i = 0; i < 4 * kSlots; ++i) { mbar_init(xbar + 8 * i, 1); mbar_init(zready + 8 * i, 1); }   // per (slot, quadrant)
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
          const int gq = tile / tok_tiles, tt = tile % tok_tiles;
          const int tok = (cur.li * c.n_seqs + cur.s) * c.W + c.q_row_begin + tt * kTileM;
#pragma unroll
          for (int p = 0; p < SM::kPanels; ++p)
            tma_load_3d(sQ + stage * SM::kQStageBytes + p * (kTileM * 128), &q_map, qfull + 8 * stage,
                        p * 64, cur.hk * c.G + gq, tok);
        }
      }
      __syncwarp();
      if (SM::kKStages == 1 && have_n) load_k(nxt);
      cur = nxt;
      have = have_n;
    }
  } else if (warp == kMmaWarp) {
    // ================================ MMA issuer ================================================
    // Two streams over the same tiles: MMA1(t) fills TMEM region A (columns 0..255) for phase 1, MMA2(t)
    // fills region B (columns 256..511) for phase 2 and runs one tile behind (phase 2 needs the row
    // statistics of the whole tile).  Each is issued as two N <= 128 halves with their own barriers.
    // The whole warp walks the segments; one elected lane issues.  Descriptor low words are base +
    // compile-time offsets: shared-memory addresses are < 2^18, so (addr >> 4) never carries out of
    // the 14-bit address field.
    constexpr uint32_t kDescHi = (uint32_t)(1024u >> 4) | (1u << 14) | (2u << 29);   // SBO | version | SWIZZLE_128B
    constexpr uint32_t kDescLo = 1u << 16;                                           // LBO (unused)
    const uint32_t b_lo = (sK >> 4) | kDescLo;
    struct Cur { long long g; int rem, n_cols; bool fresh; };
    auto advance = [&](Cur& u) {
      while (u.rem == 0 && u.g < g_end) {
        const Seg it = decode_seg(c, u.g, g_end, rank, cluster_id, n_clusters, T, tpu);
        u.g += it.t1 - it.t0;
        if (it.ok) { u.rem = it.t1 - it.t0; u.n_cols = it.n_cols; u.fresh = true; }
      }
    };
    auto issue = [&](uint32_t a_lo, uint32_t d_tmem, int nc, int hf) {
      const uint32_t idesc = make_idesc_bf16(nc);
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
    };
    Cur c1{g_begin, 0, 0, false}, c2{g_begin, 0, 0, false};
    int i1 = 0, i2 = 0, kuse = 0;
    // Whichever stream can go, goes (a strict MMA2, MMA1 alternation would couple the two phases: a late
    // phase 2 would hold back MMA1 although region A is free).  Phase 1 runs at most QS - 1 tiles ahead
    // (the Q ring); MMA2 has priority, which also keeps the single K panel moving at segment changes.
    for (;;) {
      advance(c1);
      const bool more1 = c1.rem > 0;
      if (!more1 && i2 == i1) break;
      if (i2 < i1 && mbar_test(tempty2, (i2 & 1) ^ 1)) {
        // ---- MMA2 of tile i2 (its Q stage and K panel are still resident) ----
        advance(c2);
        const int stage = i2 % QS;
        const uint32_t a_lo = ((sQ + stage * SM::kQStageBytes) >> 4) | kDescLo;
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
          mbar_wait(tempty2 + 8 * hf, (i2 & 1) ^ 1);
          tc_fence_after();
          if (elect_one()) {
            const int nc = half_cols(c2.n_cols, hf);
            if (nc > 0) issue(a_lo, tmem_base + kKeysPerCta + hf * kHalf, nc, hf);
            umma_commit(tfull2 + 8 * hf);
            if (hf == 1) {
              umma_commit(qempty + 8 * stage);           // both phases have read this Q tile
              if (c2.rem == 1) umma_commit(kempty);      // last tile of the segment: the K panel may be replaced
            }
          }
          __syncwarp();
        }
        --c2.rem; ++i2;
      } else if (more1 && i1 - i2 < QS && mbar_test(tempty1, (i1 & 1) ^ 1) &&
                 (!c1.fresh || mbar_test(kfull, kuse & 1)) && mbar_test(qfull + 8 * (i1 % QS), (i1 / QS) & 1)) {
        // ---- MMA1 of tile i1 ----
        if (c1.fresh) { mbar_wait(kfull, kuse & 1); ++kuse; c1.fresh = false; }
        const int stage = i1 % QS;
        mbar_wait(qfull + 8 * stage, (i1 / QS) & 1);
        const uint32_t a_lo = ((sQ + stage * SM::kQStageBytes) >> 4) | kDescLo;
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
          mbar_wait(tempty1 + 8 * hf, (i1 & 1) ^ 1);
          tc_fence_after();
          if (elect_one()) {
            const int nc = half_cols(c1.n_cols, hf);
            if (nc > 0) issue(a_lo, tmem_base + hf * kHalf, nc, hf);
            umma_commit(tfull1 + 8 * hf);
          }
          __syncwarp();
        }
        --c1.rem; ++i1;
      }
    }
  }
  } else if (warp >= kSWarp0) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" :: "n"(kRegsOther));
    // ================================ S warps: row statistics ======================================
    // lane = row of this quadrant.  (z, l) of the two halves -> CTA -> cluster (st.async exchange), then
    // o = Z + log2 L of the row to shared memory: phase 2 computes 2^(s c - o), the probability itself.
    const int q = warp & 3;
    int tile_iter = 0;
    for (long long g = g_begin; g < g_end;) {
      const Seg it = decode_seg(c, g, g_end, rank, cluster_id, n_clusters, T, tpu);
      g += it.t1 - it.t0;
      if (!it.ok) {
        // skipped unit: its strip must still be defined (zeros); the status word says why
        float* out = c.partial + ((long long)it.unit * c.parts + it.part) * c.n_pad;
        if (rank == 0) for (int j = threadIdx.x & 127; j < c.n_pad; j += 128) out[j] = 0.f;
        continue;
      }
      for (int tile = it.t0; tile < it.t1; ++tile, ++tile_iter) {
        const int b = tile_iter & (kSlots - 1), par = (tile_iter / kSlots) & 1;
        mbar_wait(bdone1 + 8 * b, par);
        int z_row;
        float l_row;
        {
          const uint2 s0 = rstat[(b * 2 + 0) * 128 + q * 32 + lane], s1 = rstat[(b * 2 + 1) * 128 + q * 32 + lane];
          z_row = max((int)s0.x, (int)s1.x);
          l_row = __uint_as_float(s0.y) * pow2i((int)s0.x - z_row) + __uint_as_float(s1.y) * pow2i((int)s1.x - z_row);
        }
        if (CL > 1) {
          // lane publishes its row to every peer CTA ...
          const uint32_t bar = xbar + 8 * (b * 4 + q);
          uint2* slot = xch + (size_t)(b * 4 + q) * CL * 32;
          if (lane == 0) mbar_expect_tx(bar, (CL - 1) * 32 * 8);
          __syncwarp();
          const uint32_t la = smem_u32(slot + rank * 32 + lane);
#pragma unroll
          for (int p = 0; p < CL; ++p)
            if (p != rank) st_async_b32x2(mapa(la, p), (uint32_t)z_row, __float_as_uint(l_row), mapa(bar, p));
          mbar_wait(bar, par);
          // ... and merges that row over the CTAs in rank order (identical bits on every CTA)
          int Z = z_row;
#pragma unroll
          for (int p = 0; p < CL; ++p) if (p != rank) Z = max(Z, (int)slot[p * 32 + lane].x);
          float L = 0.f;
#pragma unroll
          for (int p = 0; p < CL; ++p) {
            const uint2 v = slot[p * 32 + lane];
            L += (p == rank) ? l_row * pow2i(z_row - Z) : __uint_as_float(v.y) * pow2i((int)v.x - Z);
          }
          z_row = Z; l_row = L;
        }
        const int tok = c.q_row_begin + (tile % tok_tiles) * kTileM + q * 32 + lane;
        // rows past the window (and rows with no valid key) contribute nothing: 2^(s c - inf) = 0
        const float o = (l_row > 0.f && tok < c.W) ? (float)(z_row - kMagicBits) + __log2f(l_row) : __int_as_float(0x7f800000);
        orow[(b * 4 + q) * 32 + lane] = o;
        __syncwarp();
        if (lane == 0) mbar_arrive(zready + 8 * (b * 4 + q));
      }
    }
  } else if (warp < kP2Warp0) {
    // ================================ phase-1 warps: row statistics ====================================
    // One TMEM read of S1, nothing written back: the half is handed back to the MMA warp as soon as this
    // warp's loads have landed.  Exponentials on the FMA pipe (stats_piece).
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" :: "n"(kRegsP1));
    const int q = warp & 3, hf = (warp >> 2) & 1;       // TMEM lane quadrant; column half
    const int qd = lane & 3, lr = lane >> 2;
    const float cs = kLog2e * rsqrtf((float)D);
    const uint32_t tq = tmem_base + ((uint32_t)(q * 32) << 16) + hf * kHalf, tq_hi = tq + (16u << 16);
    auto release = [&]() {
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty1 + 8 * hf);
    };
    int tile_iter = 0;
    for (long long g = g_begin; g < g_end;) {
      const Seg it = decode_seg(c, g, g_end, rank, cluster_id, n_clusters, T, tpu);
      g += it.t1 - it.t0;
      if (!it.ok) continue;
      const int n_ch = (half_cols(it.n_cols, hf) + 63) >> 6;            // chunks of this half the MMA writes: 0 .. 2
      const int c_lo = it.c_lo, c_hi = it.c_hi;
      for (int tile = it.t0; tile < it.t1; ++tile, ++tile_iter) {
        const int b = tile_iter & (kSlots - 1);
        int zq[4];
        float lq[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) { zq[k] = kZFloor; lq[k] = 0.f; }
        mbar_wait(tfull1 + 8 * hf, tile_iter & 1);
        tc_fence_after();
        // one piece at a time (the registers go to keeping several polynomial chains in flight), the chunks in
        // a rolled loop (the unrolled kernel did not fit the instruction cache)
#pragma unroll 1
        for (int ch = 0; ch < n_ch; ++ch) {
          uint32_t r[32];
          tmem_ld_16x256b_x8(tq + ch * 64, r);
          tmem_wait_ld();
          stats_piece<0>(r, zq, lq, cs, qd, hf * kHalf + ch * 64, c_lo, c_hi);
          tmem_ld_16x256b_x8(tq_hi + ch * 64, r);
          tmem_wait_ld();
          if (ch == n_ch - 1) release();
          stats_piece<2>(r, zq, lq, cs, qd, hf * kHalf + ch * 64, c_lo, c_hi);
        }
        if (n_ch == 0) release();
        // ---- reduce-scatter over the 4 lanes of a quad (6 shuffles): lane qd ends up with row k = qd ----
        int z_row;
        float l_row;
        {
          const bool p1 = qd & 1, p2 = qd & 2;
          const int ks0 = p1 ? zq[1] : zq[0], ks1 = p1 ? zq[3] : zq[2];
          const float kl0 = p1 ? lq[1] : lq[0], kl1 = p1 ? lq[3] : lq[2];
          const int rz0 = __shfl_xor_sync(0xffffffffu, p1 ? zq[0] : zq[1], 1);
          const int rz1 = __shfl_xor_sync(0xffffffffu, p1 ? zq[2] : zq[3], 1);
          const float rl0 = __shfl_xor_sync(0xffffffffu, p1 ? lq[0] : lq[1], 1);
          const float rl1 = __shfl_xor_sync(0xffffffffu, p1 ? lq[2] : lq[3], 1);
          const int za = max(ks0, rz0), zb = max(ks1, rz1);
          const float la = kl0 * pow2i(ks0 - za) + rl0 * pow2i(rz0 - za);
          const float lb = kl1 * pow2i(ks1 - zb) + rl1 * pow2i(rz1 - zb);
          const int kz = p2 ? zb : za;
          const float kl = p2 ? lb : la;
          const int rz = __shfl_xor_sync(0xffffffffu, p2 ? za : zb, 2);
          const float rl = __shfl_xor_sync(0xffffffffu, p2 ? la : lb, 2);
          z_row = max(kz, rz);
          l_row = kl * pow2i(kz - z_row) + rl * pow2i(rz - z_row);
        }
        rstat[(b * 2 + hf) * 128 + q * 32 + lr + 8 * qd] = make_uint2((uint32_t)z_row, __float_as_uint(l_row));
        __syncwarp();
        if (lane == 0) mbar_arrive(bdone1 + 8 * b);
      }
    }
  } else {
    // ================================ phase-2 warps: scores ===========================================
    // One TMEM read of S2 (recomputed), one ex2 per element, straight into the per-thread column sums
    // (with the 16x256b load shape the sum over rows needs no transpose); nothing goes back to TMEM.
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" :: "n"(kRegsP2));
    const int q = warp & 3, hf = (warp >> 2) & 1;       // TMEM lane quadrant; column half
    const int qd = lane & 3, lr = lane >> 2;
    const float cs = kLog2e * rsqrtf((float)D);
    const uint32_t tq = tmem_base + ((uint32_t)(q * 32) << 16) + kKeysPerCta + hf * kHalf, tq_hi = tq + (16u << 16);
    uint64_t acc[2][8];                                 // column sums of this warp's two chunks over the segment
#pragma unroll
    for (int a = 0; a < 8; ++a) { acc[0][a] = 0ull; acc[1][a] = 0ull; }
    auto release = [&]() {
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty2 + 8 * hf);
    };
    int tile_iter = 0;
    for (long long g = g_begin; g < g_end;) {
      const Seg it = decode_seg(c, g, g_end, rank, cluster_id, n_clusters, T, tpu);
      g += it.t1 - it.t0;
      if (!it.ok) continue;
      const int n_ch = (half_cols(it.n_cols, hf) + 63) >> 6;            // chunks of this half the MMA writes: 0 .. 2
      float* out = c.partial + ((long long)it.unit * c.parts + it.part) * c.n_pad;
      for (int tile = it.t0; tile < it.t1; ++tile, ++tile_iter) {
        const int b = tile_iter & (kSlots - 1), par = (tile_iter / kSlots) & 1;
        mbar_wait(zready + 8 * (b * 4 + q), par);
        float o[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) o[k] = orow[(b * 4 + q) * 32 + lr + 8 * k];
        mbar_wait(tfull2 + 8 * hf, tile_iter & 1);
        tc_fence_after();
        if (n_ch > 0) {
          uint32_t ra[32], rb[32];
          tmem_ld_16x256b_x8(tq, ra);
          tmem_ld_16x256b_x8(tq_hi, rb);
          tmem_wait_ld();
          if (n_ch == 1) release();
          score_piece(ra, acc[0], cs, o[0], o[1]);
          if (n_ch > 1) tmem_ld_16x256b_x8(tq + 64, ra);
          score_piece(rb, acc[0], cs, o[2], o[3]);
          if (n_ch > 1) {
            tmem_wait_ld();
            tmem_ld_16x256b_x8(tq_hi + 64, rb);
            score_piece(ra, acc[1], cs, o[0], o[1]);
            tmem_wait_ld();
            release();
            score_piece(rb, acc[1], cs, o[2], o[3]);
          }
        } else {
          release();
        }
      }
      // ---- segment done: combine lanes (fixed order), then the 4 quadrants (fixed order), write the strip ----
#pragma unroll
      for (int ch = 0; ch < 2; ++ch) {
#pragma unroll
        for (int a = 0; a < 8; ++a) {
          float v0, v1;
          upk2(acc[ch][a], v0, v1);
          v0 += __shfl_xor_sync(0xffffffffu, v0, 4);  v1 += __shfl_xor_sync(0xffffffffu, v1, 4);
          v0 += __shfl_xor_sync(0xffffffffu, v0, 8);  v1 += __shfl_xor_sync(0xffffffffu, v1, 8);
          v0 += __shfl_xor_sync(0xffffffffu, v0, 16); v1 += __shfl_xor_sync(0xffffffffu, v1, 16);
          if (lr == 0)
            *reinterpret_cast<float2*>(&colsum[q * kKeysPerCta + hf * kHalf + ch * 64 + a * 8 + 2 * qd]) = make_float2(v0, v1);
          acc[ch][a] = 0ull;
        }
      }
      named_bar_sync(1 + hf, 128);                          // the 4 warps (quadrants) that share this half
      {
        const int x = hf * kHalf + q * 32 + lane;
        float v = 0.f;
#pragma unroll
        for (int wv = 0; wv < 4; ++wv) v += colsum[wv * kKeysPerCta + x];
        if (x >= it.c_lo && x < it.c_hi) out[rank * kKeysPerCta + x - it.off] = v;
      }
      named_bar_sync(1 + hf, 128);
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
  auto kern = score_tc2_kernel<D, CL>;
  static bool attr_done = false;
  if (!attr_done) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SM::kAlloc) != cudaSuccess)
      return tc_fail(KARA_ECUDA, "cudaFuncSetAttribute(max dynamic smem) failed");
    attr_done = true;
  }
  const int tok_tiles = (c.W - c.q_row_begin + kTileM - 1) / kTileM;
  const int tpu = tok_tiles * c.G;
  const int units = c.n_layers * c.n_seqs * c.g.n_kv_heads;
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

const char* score_tc2_error() { return g_tc_err; }

int score_tc2_launch(ScoreTcState* s, Call& c, cudaStream_t st, int* n_launches) {
  // window_q tensor map: [d][n_q_heads][layers*seqs*W tokens], box 64 x 1 x 128, 128B swizzle
  const long long key[6] = {(long long)(uintptr_t)c.window_q, c.g.d, c.n_q_heads, (long long)c.n_layers * c.n_seqs * c.W, 0, 0};
  if (s->q_ptr != c.window_q || memcmp(key, s->q_key, sizeof key) != 0) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return tc_fail(KARA_ECUDA, "cuTensorMapEncodeTiled entry point not found");
    cuuint64_t dims[3] = {(cuuint64_t)c.g.d, (cuuint64_t)c.n_q_heads, (cuuint64_t)key[3]};
    cuuint64_t strides[2] = {(cuuint64_t)c.g.d * 2, (cuuint64_t)c.g.d * 2 * c.n_q_heads};
    cuuint32_t box[3] = {64u, 1u, (cuuint32_t)kTileM};
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


