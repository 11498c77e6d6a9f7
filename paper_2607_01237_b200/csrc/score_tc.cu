// score_tc.cu — a1 (Eq. 4): A = colsum(softmax(Q_W K_{W\U}^T / sqrt(d))) on the
// 5th-generation tensor cores of sm_100a: TMA -> shared memory, tcgen05.mma -> TMEM, softmax out
// of TMEM, deterministic column sums.  DESIGN.md §Kernels/a1 has the derivation of every choice.
//
// Decomposition.  A work item is (unit, part): a unit is one (layer, sequence, KV head); a part is
// a contiguous range of the unit's query tiles; a query tile is 128 window tokens x ONE query
// head of the GQA group (rows of a row-softmax are independent, so any (token, head) -> row map
// is valid; TMA reads the rows at stride n_q_heads*d).  A thread-block cluster of CL CTAs owns an
// item; CTA r of the cluster owns the 256 key rows [256 r, 256 r + 256) of the block-aligned key
// panel (whole paged blocks are loaded, one TMA box per block and 64-element column panel; rows
// outside the compressible region [h, h+n) are masked to -inf).  Per tile and CTA:
//   S[128 x 256] = Q_tile[128 x d] . K_cta[256 x d]^T      tcgen05.mma kind::f16, bf16 in, fp32 in TMEM
//   m_i^r = max_j S_ij ;  e_ij = exp2((S_ij - m_i^r) c) (stored back to TMEM) ;  l_i^r = sum_j e_ij
//   (m^r, l^r) of the 128 rows are exchanged across the cluster through distributed shared memory:
//       m_i = max_r m_i^r ;  l_i = sum_r l_i^r exp2((m_i^r - m_i) c) ;  w_i^r = exp2((m_i^r - m_i) c) / l_i
//   acc_j += sum_i e_ij w_i^r     per-thread registers: with the 16x256b TMEM load shape a thread
//                                 holds 4 rows x 1/4 of the columns, so the column sum over ALL
//                                 tiles of the item is a plain FFMA; lanes are combined once per item.
// TMEM holds two 128 x 256 fp32 S buffers (all 512 columns): the MMA of tile t+1 runs while the
// softmax warpgroup of tile t is still reading; two softmax warpgroups alternate tiles.
//
// Warp roles (320 threads): warps 0-3 softmax WG0, 4-7 softmax WG1, 8 TMA producer, 9 MMA issuer.
// Output: partial[unit][part][j] (fp32), summed over parts in fixed order by the select kernel, so
// scores are bit-reproducible run to run (no atomics anywhere).
#include <cuda.h>

#include <cstdio>
#include <cstring>

#include "score_tc.h"

namespace kara {

namespace {

constexpr int kSoftmaxWarps = 8;
constexpr int kProducerWarp = 8;
constexpr int kMmaWarp = 9;
constexpr int kThreads = 32 * 10;
constexpr int kTileM = 128;
constexpr int kKeysPerCta = 256;
constexpr int kQStages = 3;
constexpr int kTmemCols = 512;
constexpr float kLog2e = 1.4426950408889634f;

char g_tc_err[256] = "";

// ------------------------------------------------------------------------------------------------
// PTX wrappers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "KARA_WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra KARA_DONE_%=;\n\t"
      "bra KARA_WAIT_%=;\n\t"
      "KARA_DONE_%=:\n\t}"
      :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "KARA_WAITC_%=:\n\t"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra KARA_DONEC_%=;\n\t"
      "bra KARA_WAITC_%=;\n\t"
      "KARA_DONEC_%=:\n\t}"
      :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ uint32_t mapa(uint32_t local_addr, uint32_t cta) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(cta));
  return r;
}
__device__ __forceinline__ void st_cluster_f2(uint32_t addr, float a, float b) {
  asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" :: "r"(addr), "f"(a), "f"(b) : "memory");
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" :: "r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(nthreads) : "memory");
}

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      :: "r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      :: "r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(dst_smem), "r"(ncols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(taddr), "r"(ncols) : "memory");
}
// D[tmem] (+)= A[smem desc] . B[smem desc]^T, bf16 x bf16 -> fp32
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      :: "r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}

// K-major, 128-byte-swizzled operand tile: rows at 128 B pitch, 8-row groups at 1024 B (SBO),
// descriptor version 1 (sm_100), layout type 2 = SWIZZLE_128B.  (cute/arch/mma_sm100_desc.hpp)
__device__ __forceinline__ uint64_t make_sw128_desc(uint32_t smem_addr) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr >> 4) & 0x3FFFu);       // start address, 16-byte units
  d |= (uint64_t)1u << 16;                            // leading byte offset (unused for swizzled K-major)
  d |= (uint64_t)(1024u >> 4) << 32;                  // stride byte offset: 8 rows x 128 B
  d |= (uint64_t)1u << 46;                            // descriptor version (Blackwell)
  d |= (uint64_t)2u << 61;                            // SWIZZLE_128B
  return d;
}
// instruction descriptor: fp32 accumulate, bf16 A and B, both K-major, M = 128, N = n
__device__ __forceinline__ uint32_t make_idesc_bf16(int n) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);
}

#define KARA_TMEM_REGS32(r, o)                                                                       \
  "=r"(r[o + 0]), "=r"(r[o + 1]), "=r"(r[o + 2]), "=r"(r[o + 3]), "=r"(r[o + 4]), "=r"(r[o + 5]),    \
  "=r"(r[o + 6]), "=r"(r[o + 7]), "=r"(r[o + 8]), "=r"(r[o + 9]), "=r"(r[o + 10]), "=r"(r[o + 11]),  \
  "=r"(r[o + 12]), "=r"(r[o + 13]), "=r"(r[o + 14]), "=r"(r[o + 15]), "=r"(r[o + 16]), "=r"(r[o + 17]), \
  "=r"(r[o + 18]), "=r"(r[o + 19]), "=r"(r[o + 20]), "=r"(r[o + 21]), "=r"(r[o + 22]), "=r"(r[o + 23]), \
  "=r"(r[o + 24]), "=r"(r[o + 25]), "=r"(r[o + 26]), "=r"(r[o + 27]), "=r"(r[o + 28]), "=r"(r[o + 29]), \
  "=r"(r[o + 30]), "=r"(r[o + 31])
#define KARA_TMEM_IN32(r, o)                                                                         \
  "r"(r[o + 0]), "r"(r[o + 1]), "r"(r[o + 2]), "r"(r[o + 3]), "r"(r[o + 4]), "r"(r[o + 5]),          \
  "r"(r[o + 6]), "r"(r[o + 7]), "r"(r[o + 8]), "r"(r[o + 9]), "r"(r[o + 10]), "r"(r[o + 11]),        \
  "r"(r[o + 12]), "r"(r[o + 13]), "r"(r[o + 14]), "r"(r[o + 15]), "r"(r[o + 16]), "r"(r[o + 17]),    \
  "r"(r[o + 18]), "r"(r[o + 19]), "r"(r[o + 20]), "r"(r[o + 21]), "r"(r[o + 22]), "r"(r[o + 23]),    \
  "r"(r[o + 24]), "r"(r[o + 25]), "r"(r[o + 26]), "r"(r[o + 27]), "r"(r[o + 28]), "r"(r[o + 29]),    \
  "r"(r[o + 30]), "r"(r[o + 31])

// 16 lanes x 64 columns: thread t gets, for column group i (8 columns), regs 4i+{0,1} = lane t/4,
// columns 8i + 2(t%4) + {0,1}; regs 4i+{2,3} = lane t/4 + 8, same columns.
template <int O>
__device__ __forceinline__ void tmem_ld_16x256b_x8(uint32_t taddr, uint32_t (&r)[64]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.16x256b.x8.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : KARA_TMEM_REGS32(r, O) : "r"(taddr) : "memory");
}
template <int O>
__device__ __forceinline__ void tmem_st_16x256b_x8(uint32_t taddr, const uint32_t (&r)[64]) {
  asm volatile(
      "tcgen05.st.sync.aligned.16x256b.x8.b32 [%32], "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31};"
      :: KARA_TMEM_IN32(r, O), "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// ------------------------------------------------------------------------------------------------
// shared-memory carve-up (dynamic smem, manually aligned to 1024 B for the 128B swizzle)
// ------------------------------------------------------------------------------------------------
template <int D, int CL>
struct Smem {
  static constexpr int kPanels = D / 64;
  static constexpr int kKBytes = kPanels * kKeysPerCta * 128;
  static constexpr int kQStageBytes = kPanels * kTileM * 128;
  static constexpr int kOffK = 0;
  static constexpr int kOffQ = kOffK + kKBytes;
  static constexpr int kOffColsum = kOffQ + kQStages * kQStageBytes;        // float [8][256]
  static constexpr int kOffXch = kOffColsum + kSoftmaxWarps * kKeysPerCta * 4;  // float2 [4][CL][128]
  static constexpr int kOffBars = kOffXch + 4 * CL * kTileM * 8;
  // barriers: qfull[3] qempty[3] kfull kempty tfull[2] tempty[2] xbar[4]  = 16 x 8 B
  static constexpr int kOffTmemPtr = kOffBars + 16 * 8;
  static constexpr int kBytes = kOffTmemPtr + 16;
  static constexpr int kAlloc = kBytes + 1024;   // slack for manual alignment
};

struct ItemInfo {
  int unit, part, li, s, hk, layer;
  int h, fb, off;          // window start, first key block (table index), h - fb*bs
  int c_lo, c_hi;          // this CTA's valid key columns [c_lo, c_hi) within its 256
  int n_cols;              // MMA N for this CTA: valid columns rounded up to 16 (>= 16)
  int t0, t1;              // tile range of the part
  bool ok;
};

template <int CL>
__device__ __forceinline__ ItemInfo decode_item(const Call& c, int item, int rank, int tiles_per_unit, int tiles_per_part) {
  ItemInfo it;
  it.unit = item / c.parts;
  it.part = item % c.parts;
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
  it.t0 = min(tiles_per_unit, it.part * tiles_per_part);
  it.t1 = min(tiles_per_unit, it.t0 + tiles_per_part);
  return it;
}

// ------------------------------------------------------------------------------------------------
// the kernel
// ------------------------------------------------------------------------------------------------
template <int D, int CL>
__global__ void __launch_bounds__(kThreads, 1)
score_tc_kernel(const __grid_constant__ CUtensorMap k_map, const __grid_constant__ CUtensorMap q_map,
                const Call c, int n_items, int tiles_per_unit, int tiles_per_part, int tok_tiles) {
  using SM = Smem<D, CL>;
  extern __shared__ unsigned char smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* gbase = smem_raw + (base - raw);
  const uint32_t sK = base + SM::kOffK;
  const uint32_t sQ = base + SM::kOffQ;
  float* colsum = reinterpret_cast<float*>(gbase + SM::kOffColsum);
  float2* xch = reinterpret_cast<float2*>(gbase + SM::kOffXch);
  const uint32_t bars = base + SM::kOffBars;
  const uint32_t qfull = bars, qempty = bars + 24, kfull = bars + 48, kempty = bars + 56;
  const uint32_t tfull = bars + 64, tempty = bars + 80, xbar = bars + 96;
  volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(gbase + SM::kOffTmemPtr);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rank = CL > 1 ? (int)cluster_ctarank() : 0;
  const int cluster_id = blockIdx.x / CL, n_clusters = gridDim.x / CL;

  if (threadIdx.x == 0) {
    for (int i = 0; i < kQStages; ++i) { mbar_init(qfull + 8 * i, 1); mbar_init(qempty + 8 * i, 1); }
    mbar_init(kfull, 1);
    mbar_init(kempty, 1);
    for (int i = 0; i < 2; ++i) { mbar_init(tfull + 8 * i, 1); mbar_init(tempty + 8 * i, 1); }
    for (int i = 0; i < 4; ++i) mbar_init(xbar + 8 * i, 4 * CL);   // one arrive per softmax warp per CTA
    fence_barrier_init();
  }
  if (warp == kMmaWarp) tmem_alloc(smem_u32((const void*)tmem_ptr), kTmemCols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (CL > 1) cluster_sync_all();
  const uint32_t tmem_base = *tmem_ptr;

  if (warp == kProducerWarp) {
    // ================================ TMA producer ==============================================
    int q_iter = 0, k_iter = 0;
    const int blocks_per_cta = kKeysPerCta >> c.g.bs_log2;   // <= 16: one block per lane
    for (int item = cluster_id; item < n_items; item += n_clusters) {
      const ItemInfo it = decode_item<CL>(c, item, rank, tiles_per_unit, tiles_per_part);
      if (!it.ok || it.t0 >= it.t1) continue;
      // ---- K panel of this CTA: whole blocks, skipped if they hold no compressible key ----
      mbar_wait(kempty, (k_iter & 1) ^ 1);
      ++k_iter;
      int my_bytes = 0;
      int my_blk = -1, my_row = 0;
      if (lane < blocks_per_cta) {
        const int lb = lane;
        const int row0 = lb << c.g.bs_log2;                       // first panel row of this block in the CTA
        if (row0 < it.c_hi && row0 + c.g.bs > it.c_lo) {          // block intersects the valid columns
          const int tbl = it.fb + rank * blocks_per_cta + lb;
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
      if (lane == 0) mbar_expect_tx(kfull, (uint32_t)tot);
      __syncwarp();
      if (my_blk >= 0) {
        const long long grow = (((long long)it.layer * c.g.num_blocks + my_blk) * c.g.n_kv_heads + it.hk) << c.g.bs_log2;
#pragma unroll
        for (int p = 0; p < SM::kPanels; ++p)
          tma_load_2d(sK + p * (kKeysPerCta * 128) + my_row * 128, &k_map, kfull, p * 64, (int)grow);
      }
      // ---- Q tiles ----
      if (lane == 0) {
        for (int tile = it.t0; tile < it.t1; ++tile, ++q_iter) {
          const int stage = q_iter % kQStages, use = q_iter / kQStages;
          mbar_wait(qempty + 8 * stage, (use & 1) ^ 1);
          mbar_expect_tx(qfull + 8 * stage, SM::kQStageBytes);
          const int g = tile / tok_tiles, tt = tile % tok_tiles;
          const int tok = (it.li * c.n_seqs + it.s) * c.W + c.q_row_begin + tt * kTileM;
#pragma unroll
          for (int p = 0; p < SM::kPanels; ++p)
            tma_load_3d(sQ + stage * SM::kQStageBytes + p * (kTileM * 128), &q_map, qfull + 8 * stage,
                        p * 64, it.hk * c.G + g, tok);
        }
      }
      __syncwarp();
    }
  } else if (warp == kMmaWarp) {
    // ================================ MMA issuer ================================================
    int q_iter = 0, k_iter = 0, tile_iter = 0;
    for (int item = cluster_id; item < n_items; item += n_clusters) {
      const ItemInfo it = decode_item<CL>(c, item, rank, tiles_per_unit, tiles_per_part);
      if (!it.ok || it.t0 >= it.t1) continue;
      const uint32_t idesc = make_idesc_bf16(it.n_cols);
      if (lane == 0) {
        mbar_wait(kfull, k_iter & 1);
        for (int tile = it.t0; tile < it.t1; ++tile, ++q_iter, ++tile_iter) {
          const int stage = q_iter % kQStages, quse = q_iter / kQStages;
          const int buf = tile_iter & 1, tuse = tile_iter >> 1;
          mbar_wait(qfull + 8 * stage, quse & 1);
          mbar_wait(tempty + 8 * buf, (tuse & 1) ^ 1);
          tc_fence_after();
          const uint32_t d_tmem = tmem_base + buf * kKeysPerCta;
#pragma unroll
          for (int p = 0; p < SM::kPanels; ++p) {
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
              const uint64_t ad = make_sw128_desc(sQ + stage * SM::kQStageBytes + p * (kTileM * 128) + ks * 32);
              const uint64_t bd = make_sw128_desc(sK + p * (kKeysPerCta * 128) + ks * 32);
              umma_bf16(d_tmem, ad, bd, idesc, (p | ks) != 0);
            }
          }
          umma_commit(qempty + 8 * stage);   // Q stage reusable once these MMAs have read it
          umma_commit(tfull + 8 * buf);      // S tile complete
        }
        umma_commit(kempty);                 // K panel reusable
      }
      ++k_iter;
      __syncwarp();
    }
  } else {
    // ================================ softmax warpgroups =========================================
    const int wg = warp >> 2, wq = warp & 3;
    const int qd = lane & 3, lr = lane >> 2;            // column pair within a group of 8; row within 8
    const float cs = kLog2e * rsqrtf((float)D);
    const uint32_t lane_base = (uint32_t)(wq * 32) << 16;
    float acc[64];
#pragma unroll
    for (int a = 0; a < 64; ++a) acc[a] = 0.f;
    int tile_iter = 0, my_tiles = 0;
    for (int item = cluster_id; item < n_items; item += n_clusters) {
      const ItemInfo it = decode_item<CL>(c, item, rank, tiles_per_unit, tiles_per_part);
      float* out = c.partial + ((long long)it.unit * c.parts + it.part) * c.n_pad;
      if (!it.ok || it.t0 >= it.t1) {
        // skipped item: its strip of partial sums must still be defined (zeros)
        if (rank == 0) for (int j = threadIdx.x; j < c.n_pad; j += 32 * kSoftmaxWarps) out[j] = 0.f;
        continue;
      }
      const int n_chunks = (it.n_cols + 63) >> 6;
      for (int tile = it.t0; tile < it.t1; ++tile, ++tile_iter) {
        if ((tile_iter & 1) != wg) continue;
        const int buf = wg, use = my_tiles;
        ++my_tiles;
        const int tt = tile % tok_tiles;
        const int tok0 = c.q_row_begin + tt * kTileM;
        mbar_wait(tfull + 8 * buf, (tile_iter >> 1) & 1);
        tc_fence_after();
        const uint32_t taddr = tmem_base + lane_base + buf * kKeysPerCta;
        uint32_t r[64];

        auto load_chunk = [&](int ch) {
          tmem_ld_16x256b_x8<0>(taddr + ch * 64, r);
          tmem_ld_16x256b_x8<32>(taddr + (16u << 16) + ch * 64, r);
          tmem_wait_ld();
        };
        auto mask_chunk = [&](int ch) {
          const int cb = ch * 64;
          if (cb >= it.c_lo && cb + 64 <= it.c_hi) return;
#pragma unroll
          for (int i = 0; i < 8; ++i) {
#pragma unroll
            for (int j = 0; j < 2; ++j) {
              const int col = cb + 8 * i + 2 * qd + j;
              const bool v = (col >= it.c_lo) && (col < it.c_hi);
              if (!v) {
                r[4 * i + j] = 0xff800000u; r[4 * i + 2 + j] = 0xff800000u;
                r[32 + 4 * i + j] = 0xff800000u; r[32 + 4 * i + 2 + j] = 0xff800000u;
              }
            }
          }
        };

        // ---- pass A: row maxima over this CTA's valid columns ----
        float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
        for (int ch = 0; ch < n_chunks; ++ch) {
          load_chunk(ch);
          mask_chunk(ch);
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            mx[0] = fmaxf(mx[0], fmaxf(__uint_as_float(r[4 * i]), __uint_as_float(r[4 * i + 1])));
            mx[1] = fmaxf(mx[1], fmaxf(__uint_as_float(r[4 * i + 2]), __uint_as_float(r[4 * i + 3])));
            mx[2] = fmaxf(mx[2], fmaxf(__uint_as_float(r[32 + 4 * i]), __uint_as_float(r[32 + 4 * i + 1])));
            mx[3] = fmaxf(mx[3], fmaxf(__uint_as_float(r[32 + 4 * i + 2]), __uint_as_float(r[32 + 4 * i + 3])));
          }
        }
        float ms[4];   // local row max in the exp2 domain; 0 stands in for "no valid key in this CTA"
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          mx[k] = fmaxf(mx[k], __shfl_xor_sync(0xffffffffu, mx[k], 1));
          mx[k] = fmaxf(mx[k], __shfl_xor_sync(0xffffffffu, mx[k], 2));
          ms[k] = (mx[k] == -INFINITY) ? 0.f : mx[k] * cs;
        }
        // ---- pass B: e = exp2(s c - m c), row sums, e written back in place ----
        float ls[4] = {0.f, 0.f, 0.f, 0.f};
        for (int ch = 0; ch < n_chunks; ++ch) {
          load_chunk(ch);
          mask_chunk(ch);
#pragma unroll
          for (int i = 0; i < 8; ++i) {
#pragma unroll
            for (int j = 0; j < 2; ++j) {
              const float e0 = ex2(fmaf(__uint_as_float(r[4 * i + j]), cs, -ms[0]));
              const float e1 = ex2(fmaf(__uint_as_float(r[4 * i + 2 + j]), cs, -ms[1]));
              const float e2 = ex2(fmaf(__uint_as_float(r[32 + 4 * i + j]), cs, -ms[2]));
              const float e3 = ex2(fmaf(__uint_as_float(r[32 + 4 * i + 2 + j]), cs, -ms[3]));
              ls[0] += e0; ls[1] += e1; ls[2] += e2; ls[3] += e3;
              r[4 * i + j] = __float_as_uint(e0); r[4 * i + 2 + j] = __float_as_uint(e1);
              r[32 + 4 * i + j] = __float_as_uint(e2); r[32 + 4 * i + 2 + j] = __float_as_uint(e3);
            }
          }
          tmem_st_16x256b_x8<0>(taddr + ch * 64, r);
          tmem_st_16x256b_x8<32>(taddr + (16u << 16) + ch * 64, r);
        }
        tmem_wait_st();
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          ls[k] += __shfl_xor_sync(0xffffffffu, ls[k], 1);
          ls[k] += __shfl_xor_sync(0xffffffffu, ls[k], 2);
        }
        // local "max" that is honest about emptiness for the exchange
        float mloc[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) mloc[k] = (mx[k] == -INFINITY) ? -INFINITY : ms[k];

        // ---- row weights w_i: cluster-wide softmax normalisation ----
        float w[4];
        if (CL == 1) {
#pragma unroll
          for (int k = 0; k < 4; ++k) w[k] = ls[k] > 0.f ? 1.f / ls[k] : 0.f;
        } else {
          const int slot = wg * 2 + (use & 1);
          float2* my_slot = xch + (size_t)slot * CL * kTileM;
          if (qd == 0) {
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              const int row = wq * 32 + lr + 8 * k;
              const uint32_t la = smem_u32(my_slot + (size_t)rank * kTileM + row);
#pragma unroll
              for (int p = 0; p < CL; ++p) st_cluster_f2(mapa(la, p), mloc[k], ls[k]);
            }
          }
          __syncwarp();
          if (lane == 0) {
            asm volatile("fence.acq_rel.cluster;" ::: "memory");
#pragma unroll
            for (int p = 0; p < CL; ++p) mbar_arrive_remote(mapa(xbar + 8 * slot, p));
          }
          mbar_wait_cluster(xbar + 8 * slot, (use >> 1) & 1);
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const int row = wq * 32 + lr + 8 * k;
            float M = -INFINITY;
            float2 v[CL];
#pragma unroll
            for (int p = 0; p < CL; ++p) { v[p] = my_slot[(size_t)p * kTileM + row]; M = fmaxf(M, v[p].x); }
            float l = 0.f;
#pragma unroll
            for (int p = 0; p < CL; ++p) l += (v[p].x == -INFINITY) ? 0.f : v[p].y * ex2(v[p].x - M);
            w[k] = (mloc[k] == -INFINITY || !(l > 0.f)) ? 0.f : ex2(mloc[k] - M) / l;
          }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k)
          if (tok0 + wq * 32 + lr + 8 * k >= c.W) w[k] = 0.f;       // rows past the window contribute nothing

        // ---- pass C: acc_j += sum_i e_ij w_i ----
        for (int ch = 0; ch < n_chunks; ++ch) {
          load_chunk(ch);
          switch (ch) {   // compile-time accumulator indices
#define KARA_ACC_CHUNK(CH)                                                                             \
            case CH:                                                                                   \
              _Pragma("unroll") for (int i = 0; i < 8; ++i) {                                          \
                _Pragma("unroll") for (int j = 0; j < 2; ++j) {                                        \
                  float a = acc[CH * 16 + 2 * i + j];                                                  \
                  a = fmaf(__uint_as_float(r[4 * i + j]), w[0], a);                                    \
                  a = fmaf(__uint_as_float(r[4 * i + 2 + j]), w[1], a);                                \
                  a = fmaf(__uint_as_float(r[32 + 4 * i + j]), w[2], a);                               \
                  a = fmaf(__uint_as_float(r[32 + 4 * i + 2 + j]), w[3], a);                           \
                  acc[CH * 16 + 2 * i + j] = a;                                                        \
                }                                                                                      \
              }                                                                                        \
              break;
            KARA_ACC_CHUNK(0) KARA_ACC_CHUNK(1) KARA_ACC_CHUNK(2) KARA_ACC_CHUNK(3)
#undef KARA_ACC_CHUNK
          }
        }
        // ---- release the TMEM buffer to the MMA warp ----
        tc_fence_before();
        named_bar_sync(1 + wg, 128);
        if ((threadIdx.x & 127) == 0) mbar_arrive(tempty + 8 * buf);
      }

      // ---- item done: combine lanes (fixed order), then warps (fixed order), write the strip ----
#pragma unroll
      for (int a = 0; a < 64; ++a) {
        float v = acc[a];
        v += __shfl_xor_sync(0xffffffffu, v, 4);
        v += __shfl_xor_sync(0xffffffffu, v, 8);
        v += __shfl_xor_sync(0xffffffffu, v, 16);
        if (lr == 0) colsum[warp * kKeysPerCta + (a >> 4) * 64 + ((a & 15) >> 1) * 8 + 2 * qd + (a & 1)] = v;
        acc[a] = 0.f;
      }
      named_bar_sync(3, 32 * kSoftmaxWarps);
      {
        const int x = threadIdx.x;   // 0..255: one column each
        float v = 0.f;
#pragma unroll
        for (int wv = 0; wv < kSoftmaxWarps; ++wv) v += colsum[wv * kKeysPerCta + x];
        if (x >= it.c_lo && x < it.c_hi) out[rank * kKeysPerCta + x - it.off] = v;
      }
      named_bar_sync(3, 32 * kSoftmaxWarps);
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
  static bool attr_done = false;
  if (!attr_done) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SM::kAlloc) != cudaSuccess)
      return tc_fail(KARA_ECUDA, "cudaFuncSetAttribute(max dynamic smem) failed");
    attr_done = true;
  }
  const int tok_tiles = (c.W - c.q_row_begin + kTileM - 1) / kTileM;
  const int tiles_per_unit = tok_tiles * c.G;
  const int units = c.n_layers * c.n_seqs * c.g.n_kv_heads;

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
  // split units into parts when that fills the last wave better (tail effect)
  int best_parts = 1;
  double best_eff = -1.0;
  for (int parts = 1; parts <= 4 && parts <= tiles_per_unit; parts *= 2) {
    const double items = (double)units * parts;
    const double rounds = items / max_clusters;
    const double eff = rounds / (double)((long long)((items + max_clusters - 1) / max_clusters)) - 0.015 * (parts - 1);
    if (eff > best_eff + 1e-9) { best_eff = eff; best_parts = parts; }
  }
  c.parts = best_parts;
  const int tiles_per_part = (tiles_per_unit + c.parts - 1) / c.parts;
  const long long n_items = (long long)units * c.parts;
  const int n_clusters = (int)(n_items < max_clusters ? n_items : max_clusters);
  cfg.gridDim = dim3(CL * n_clusters);

  CUtensorMap kmap, qmap;
  memcpy(&kmap, s->k_map, sizeof kmap);
  memcpy(&qmap, s->q_map, sizeof qmap);
  cudaError_t e = cudaLaunchKernelEx(&cfg, kern, kmap, qmap, (const Call)c, (int)n_items, tiles_per_unit,
                                     tiles_per_part, tok_tiles);
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
