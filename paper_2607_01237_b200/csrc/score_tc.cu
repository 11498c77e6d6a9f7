// score_tc.cu — a1 (Eq. 4): A = colsum(softmax(Q_W K_{W\\U}^T / sqrt(d))) on the
// 5th-generation tensor cores of sm_100a: TMA -> shared memory, tcgen05.mma -> TMEM, softmax out
// of TMEM, deterministic column sums.  DESIGN.md §Kernels/a1 has the derivation of every choice.
//
// Decomposition.  A unit is one (layer, sequence, KV head).  A query tile is 128 window tokens x
// ONE query head of the GQA group (rows of a row-softmax are independent, so any (token, head) ->
// row map is valid; TMA reads the rows at stride n_q_heads*d).  All T = units * tiles_per_unit
// tiles of the launch form one sequence that is cut into n_clusters contiguous, equally long
// ranges (perfect balance; a range crosses unit boundaries, the part of a unit inside a range is
// a "segment").  A thread-block cluster of CL CTAs owns a range; CTA r of the cluster owns the
// 256 key rows [256 r, 256 r + 256) of the block-aligned key panel (whole paged blocks are
// loaded, one TMA box per block and 64-element column panel; rows outside the compressible
// region [h, h+n) are masked to -inf).  Per tile and CTA:
//   S[128 x 256] = Q_tile[128 x d] . K_cta[256 x d]^T      tcgen05.mma kind::f16, bf16 in, fp32 in TMEM,
//       issued as two N <= 128 halves, each with its own full / empty barrier, so a half is
//       refilled as soon as its column sums have been taken.
//   The softmax is split over SPECIALISED warps (the v2 kernel ran both passes in the same warps
//   and was bound by the latency of its own dependency chain, 2 warps per sub-partition):
//   B warps (16: TMEM lane quadrant q x 64-column chunk cq) — pass B, the only MUFU work.  One TMEM
//       read, one write: a thread holds 2 rows x 16 columns per piece (two pieces per tile); it shifts
//       by ITS OWN maximum of those 16 logits, rounded to an integer z (log2 domain):
//       e = exp2(s c - z), written back in place; l += e.  No separate max pass, no shuffles inside
//       the pass.  Per tile a 6-shuffle reduce-scatter merges (z, l) over the 4 lanes of a row; shifts
//       per (thread, row, chunk) (int16) and (z, l) per (row, chunk) go to shared memory; B warps
//       never wait for anything but the next S half.
//   C warps (4: one per lane quadrant) — statistics and pass C.  (z, l) of a row are merged over
//       the four chunks and the CL CTAs with exact power-of-two rescaling built by integer
//       arithmetic (no MUFU); across CTAs with st.async + a transaction-count mbarrier per
//       (buffer, quadrant) — no fence, no cluster barrier.  w_(row,chunk) = 2^(z - Z_row) / L_row.
//       pass C (one TMEM read):  acc_j += sum_i e_ij w_i  in per-thread registers: with the 16x256b
//       TMEM load shape the column sum over ALL tiles of a segment is a plain packed FFMA2;
//       lanes are combined once per segment.
// TMEM holds two 128 x 256 fp32 S buffers (all 512 columns).  The K panel is double-buffered so a
// segment change costs no bubble.
//
// Warp roles (768 threads): warps 0-15 B (q = warp & 3, cq = warp >> 2), 16-19 C (q = warp & 3),
// 20 TMA producer, 21 MMA issuer, 22-23 idle (they complete the warpgroup whose registers
// setmaxnreg hands to the C warps).
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
constexpr int kThreads = 32 * 24;             // 6 warpgroups (setmaxnreg works per warpgroup); warps 22, 23 idle
// registers: 768 x 80 at launch; setmaxnreg only moves registers inside that allocation:
// 4 x 72 (B) + 152 (C) + 40 (producer, MMA, idle) = 6 x 80
constexpr int kRegsB = 72, kRegsC = 152, kRegsOther = 40;
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
  static constexpr int kOffZc = kOffColsum + 4 * kKeysPerCta * 4;        // short [2 bufs][4 q][4 chunks][4 rows][32 lanes] (unbiased shifts)
  static constexpr int kOffRstat = kOffZc + 2 * 4 * 4 * 4 * 32 * 2;      // uint2 [2 bufs][4 chunks][128 rows]
  static constexpr int kOffXch = kOffRstat + 2 * 4 * 128 * 8;            // uint2 [2 bufs][4 q][CL][32]
  static constexpr int kOffBars = kOffXch + 2 * 4 * CL * 32 * 8;
  // barriers: qfull[2] qempty[2] kfull[2] kempty[2] tfull[2][2] tempty[2][2] bdone[2] xbar[2][4] = 26 x 8 B
  static constexpr int kOffTmemPtr = kOffBars + 26 * 8;
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

// ---- pass B on one piece: 2 rows (K0, K0+1) x 16 columns of chunk CH (of this half) -----------------
// r[4i+j] = row K0, r[4i+2+j] = row K0+1, column col0 + 8 i + 2 qd + j of the CTA's 256; e gets the
// exponentials in the same layout.  Online softmax with exact power-of-two rescaling: the shift of
// this (row, chunk) is the running maximum z = max(z_run, round(m c)) of the thread's integer shifts
// (log2 domain), so e <= 2^0.5; l_run is rescaled by 2^(z_old - z) built from the exponent field (no
// MUFU).  Shifts are biased ints (see kZFloor); a fully masked piece has m = -inf -> as_int(t) < 0
// -> z = floor / z_run, e = 0.
template <int CH, int K0, bool RAGGED>
__device__ __forceinline__ void pass_b_body(const uint32_t (&rin)[32], uint32_t (&e)[32], int (&zc)[2][4],
                                            int (&zrun)[4], float (&lrun)[4], float cs, int qd, int col0,
                                            int c_lo, int c_hi) {
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
  int z0, z1;
  float l0s, l1s;
  if (CH == 0) {                                 // first chunk of the tile: nothing accumulated yet
    z0 = max(kZFloor, __float_as_int(t0)); z1 = max(kZFloor, __float_as_int(t1));
    l0s = 0.f; l1s = 0.f;
  } else {
    z0 = max(zrun[K0], __float_as_int(t0)); z1 = max(zrun[K0 + 1], __float_as_int(t1));
    l0s = lrun[K0] * pow2i(zrun[K0] - z0); l1s = lrun[K0 + 1] * pow2i(zrun[K0 + 1] - z1);
  }
  zrun[K0] = z0; zrun[K0 + 1] = z1;
  zc[CH][K0] = z0; zc[CH][K0 + 1] = z1;
  const float nz0 = kMagic - __int_as_float(z0), nz1 = kMagic - __int_as_float(z1);   // = -z, exact
  const uint64_t cs2 = pk2(cs, cs), nz0_2 = pk2(nz0, nz0), nz1_2 = pk2(nz1, nz1);
  uint64_t l0 = pk2(l0s, 0.f), l1 = pk2(l1s, 0.f);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    // kPolyMask: column groups whose exponentials run on the FMA pipe (never on a ragged chunk,
    // where masked columns must come out as exact zeros)
    const bool poly = !RAGGED && ((kPolyMask >> i) & 1);
    float a, b;
    if (poly) exp2_poly2(fma2(pk2(x[4 * i], x[4 * i + 1]), cs2, nz0_2), a, b);
    else { upk2(fma2(pk2(x[4 * i], x[4 * i + 1]), cs2, nz0_2), a, b); a = ex2(a); b = ex2(b); }
    l0 = add2(l0, pk2(a, b));
    e[4 * i] = __float_as_uint(a); e[4 * i + 1] = __float_as_uint(b);
    if (poly) exp2_poly2(fma2(pk2(x[4 * i + 2], x[4 * i + 3]), cs2, nz1_2), a, b);
    else { upk2(fma2(pk2(x[4 * i + 2], x[4 * i + 3]), cs2, nz1_2), a, b); a = ex2(a); b = ex2(b); }
    l1 = add2(l1, pk2(a, b));
    e[4 * i + 2] = __float_as_uint(a); e[4 * i + 3] = __float_as_uint(b);
  }
  float a, b;
  upk2(l0, a, b); lrun[K0] = a + b;
  upk2(l1, a, b); lrun[K0 + 1] = a + b;
}
// two copies of the body, so that the common (no ragged edge) path carries no select and no register copies
template <int CH, int K0>
__device__ __forceinline__ void pass_b_piece(const uint32_t (&rin)[32], uint32_t (&e)[32], int (&zc)[2][4],
                                             int (&zrun)[4], float (&lrun)[4], float cs, int qd, int col0,
                                             int c_lo, int c_hi) {
  if (col0 >= c_lo && col0 + 64 <= c_hi)        // warp-uniform: false only on the ragged first / last chunk
    pass_b_body<CH, K0, false>(rin, e, zc, zrun, lrun, cs, qd, col0, c_lo, c_hi);
  else
    pass_b_body<CH, K0, true>(rin, e, zc, zrun, lrun, cs, qd, col0, c_lo, c_hi);
}

// ---- pass C on one piece: acc[C*8 + i] (columns 64 C + 8i+2qd+{0,1}) += e(row) * w(row, chunk) -------
template <int C, int K0>
__device__ __forceinline__ void pass_c_piece(const uint32_t (&r)[32], uint64_t (&acc)[32], const float (&w)[4][4]) {
  const uint64_t w0 = pk2(w[C][K0], w[C][K0]), w1 = pk2(w[C][K0 + 1], w[C][K0 + 1]);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    uint64_t a = acc[C * 8 + i];
    a = fma2(pk2u(r[4 * i], r[4 * i + 1]), w0, a);
    a = fma2(pk2u(r[4 * i + 2], r[4 * i + 3]), w1, a);
    acc[C * 8 + i] = a;
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
  short* zcs = reinterpret_cast<short*>(gbase + SM::kOffZc);
  uint2* rstat = reinterpret_cast<uint2*>(gbase + SM::kOffRstat);
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
    for (int i = 0; i < 2; ++i) mbar_init(bdone + 8 * i, kBWarps);  // one arrive per B warp
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
      const int n_chunks = (it.n_cols + 63) >> 6;                       // 1 .. 4
      for (int tile = it.t0; tile < it.t1; ++tile, ++tile_iter) {
        const int b = tile_iter & 1, par = (tile_iter >> 1) & 1;
        mbar_wait(bdone + 8 * b, par);
        // ---- row statistics (lane = row of this quadrant): two halves -> CTA -> cluster ----
        int z_row;
        float l_row;
        {
          uint2 sc[4];
#pragma unroll
          for (int ch = 0; ch < 4; ++ch) sc[ch] = rstat[(b * 4 + ch) * 128 + q * 32 + lane];
          z_row = max(max((int)sc[0].x, (int)sc[1].x), max((int)sc[2].x, (int)sc[3].x));
          l_row = 0.f;
#pragma unroll
          for (int ch = 0; ch < 4; ++ch) l_row += __uint_as_float(sc[ch].y) * pow2i((int)sc[ch].x - z_row);
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
        const float inv_row = (l_row > 0.f && tok < c.W) ? __fdividef(1.f, l_row) : 0.f;   // rows past the window contribute nothing
        float w[4][4];
        {
          const short* zt = zcs + (size_t)((b * 4 + q) * 16) * 32 + lane;
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const int zf = __shfl_sync(0xffffffffu, z_row, lr + 8 * k) - kMagicBits;
            const float iv = __shfl_sync(0xffffffffu, inv_row, lr + 8 * k);
#pragma unroll
            for (int ch = 0; ch < 4; ++ch)
              w[ch][k] = ch < n_chunks ? iv * pow2i(zt[(ch * 4 + k) * 32] - zf) : 0.f;
          }
        }
        // ---- pass C: acc_j += sum_i e_ij w_i ; TMEM loads double buffered; halves released early ----
        tc_fence_after();
        const uint32_t ta = tq + b * kKeysPerCta, ta_hi = ta + (16u << 16);
        uint32_t ra[32], rb[32];
        tmem_ld_16x256b_x8(ta, ra);
        tmem_wait_ld();
        tmem_ld_16x256b_x8(ta_hi, rb);
        pass_c_piece<0, 0>(ra, acc, w);
        tmem_wait_ld();
        if (n_chunks > 1) tmem_ld_16x256b_x8(ta + 64, ra);
        pass_c_piece<0, 2>(rb, acc, w);
        if (n_chunks > 1) {
          tmem_wait_ld();
          tmem_ld_16x256b_x8(ta_hi + 64, rb);
          pass_c_piece<1, 0>(ra, acc, w);
          tmem_wait_ld();
          if (n_chunks > 2) tmem_ld_16x256b_x8(ta + 128, ra);
          pass_c_piece<1, 2>(rb, acc, w);
        }
        // half 0 has been read completely: the MMA may refill it
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty + 8 * (b * 2 + 0));
        if (n_chunks > 2) {
          tmem_wait_ld();
          tmem_ld_16x256b_x8(ta_hi + 128, rb);
          pass_c_piece<2, 0>(ra, acc, w);
          tmem_wait_ld();
          if (n_chunks > 3) tmem_ld_16x256b_x8(ta + 192, ra);
          pass_c_piece<2, 2>(rb, acc, w);
          if (n_chunks > 3) {
            tmem_wait_ld();
            tmem_ld_16x256b_x8(ta_hi + 192, rb);
            pass_c_piece<3, 0>(ra, acc, w);
            tmem_wait_ld();
            pass_c_piece<3, 2>(rb, acc, w);
          }
        }
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
    const int q = warp & 3, cq = warp >> 2, hf = cq >> 1;   // TMEM lane quadrant; 64-column chunk; MMA half of the chunk
    const int qd = lane & 3, lr = lane >> 2;
    const float cs = kLog2e * rsqrtf((float)D);
    const uint32_t tq = tmem_base + ((uint32_t)(q * 32) << 16) + cq * 64;
    int tile_iter = 0;
    for (long long g = g_begin; g < g_end;) {
      const Seg it = decode_seg(c, g, g_end, rank, cluster_id, n_clusters, T, tpu);
      g += it.t1 - it.t0;
      if (!it.ok) continue;
      const bool active = cq * 64 < it.n_cols;              // the MMA writes this chunk
      const int c_lo = it.c_lo, c_hi = it.c_hi;
      for (int tile = it.t0; tile < it.t1; ++tile, ++tile_iter) {
        const int b = tile_iter & 1, par = (tile_iter >> 1) & 1;
        int zc[2][4], zq[4];
        float lq[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) { zq[k] = kZFloor; lq[k] = 0.f; zc[0][k] = kZFloor; }
        mbar_wait(tfull + 8 * (b * 2 + hf), par);
        tc_fence_after();
        if (active) {
          // ---- pass B: e = 2^(s c - z) in place; z per (thread, row), (z, l) per row ----
          const uint32_t ta = tq + b * kKeysPerCta, ta_hi = ta + (16u << 16);
          uint32_t ra[32], rb[32], e[32];
          tmem_ld_16x256b_x8(ta, ra);
          tmem_wait_ld();
          tmem_ld_16x256b_x8(ta_hi, rb);
          pass_b_piece<0, 0>(ra, e, zc, zq, lq, cs, qd, cq * 64, c_lo, c_hi);
          tmem_st_16x256b_x8(ta, e);
          tmem_wait_ld();
          pass_b_piece<0, 2>(rb, e, zc, zq, lq, cs, qd, cq * 64, c_lo, c_hi);
          tmem_st_16x256b_x8(ta_hi, e);
        }
        // ---- row statistics of this chunk: quad -> row; shifts and (z, l) to shared memory ----
        {
          short* zt = zcs + (size_t)((b * 4 + q) * 16 + cq * 4) * 32 + lane;
#pragma unroll
          for (int k = 0; k < 4; ++k) zt[k * 32] = (short)(zc[0][k] - kMagicBits);
        }
        // reduce-scatter over the 4 lanes of a quad: lane qd ends up with row k = qd (6 shuffles)
        int z_row;
        float l_row;
        {
          const bool p1 = qd & 1, p2 = qd & 2;
          // step 1 (lane ^ 1): keep rows {p1, p1 + 2}, hand the other two over
          const int ks0 = p1 ? zq[1] : zq[0], ks1 = p1 ? zq[3] : zq[2];
          const float kl0 = p1 ? lq[1] : lq[0], kl1 = p1 ? lq[3] : lq[2];
          const int rz0 = __shfl_xor_sync(0xffffffffu, p1 ? zq[0] : zq[1], 1);
          const int rz1 = __shfl_xor_sync(0xffffffffu, p1 ? zq[2] : zq[3], 1);
          const float rl0 = __shfl_xor_sync(0xffffffffu, p1 ? lq[0] : lq[1], 1);
          const float rl1 = __shfl_xor_sync(0xffffffffu, p1 ? lq[2] : lq[3], 1);
          const int za = max(ks0, rz0), zb = max(ks1, rz1);
          const float la = kl0 * pow2i(ks0 - za) + rl0 * pow2i(rz0 - za);
          const float lb = kl1 * pow2i(ks1 - zb) + rl1 * pow2i(rz1 - zb);
          // step 2 (lane ^ 2): keep row p1 + 2 p2 = qd
          const int kz = p2 ? zb : za;
          const float kl = p2 ? lb : la;
          const int rz = __shfl_xor_sync(0xffffffffu, p2 ? za : zb, 2);
          const float rl = __shfl_xor_sync(0xffffffffu, p2 ? la : lb, 2);
          z_row = max(kz, rz);
          l_row = kl * pow2i(kz - z_row) + rl * pow2i(rz - z_row);
        }
        rstat[(b * 4 + cq) * 128 + q * 32 + lr + 8 * qd] = make_uint2((uint32_t)z_row, __float_as_uint(l_row));
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

bool score_tc_supported(const ScoreTcState& s, const Call& c) {
  if (!s.ready) return false;
  if (c.g.d != 64 && c.g.d != 128) return false;
  if (c.g.bs > kKeysPerCta) return false;
  if (cluster_size_for(c) == 0) return false;
  const unsigned long long toks = (unsigned long long)c.n_layers * c.n_seqs * c.W;
  if (toks >= (1ull << 31)) return false;
  return true;
}

int score_tc_launch(ScoreTcState* s, Call& c, cudaStream_t st, int* n_launches) {
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

