// qproj.cu — the window-query producer (App. C.2: at each compression the window's
// query states are recomputed — "we compute only the query projections, ..."):
//     q[t][h][:] = RoPE_{pos[t]}( hidden[t][:] . Wq[h d + :][:]^T )          bf16 in, fp32 accumulate, bf16 out
// written directly in the [token][q head][d] layout kara_compress_window reads (reading G19: rotate-half pairing,
// no bias, no q-norm).  A plain tcgen05 GEMM with the rotary embedding, the bf16 rounding and the layout fused into its epilogue:
//   persistent CTAs (one per SM) over 128 x 256 output tiles (2 heads at d = 128), K in steps of 64 through a 4-stage
//   TMA ring (128B swizzle, K-major A and B), tcgen05.mma kind::f16 M = 128, N = 256, fp32 accumulators double buffered in
//   TMEM (2 x 256 columns) so the epilogue of a tile runs under the MMAs of the next;
//   warp 0 TMA producer, warp 1 MMA issuer, warps 2-5 epilogue (a thread = an output row; TMEM read with 32x32b.x8
//   loads, the fast shape of DESIGN.md §6): columns c and c + d/2 of a head are rotated by the angle pos * theta^(-2c/d),
//   cos / sin from two small tables (angle addition over pos = 256 hi + lo, built in double precision per call).
#include "score_tc_ptx.cuh"

namespace kara {

namespace {

constexpr int kQM = 128, kQN = 256, kQK = 64, kQStages = 4;
constexpr int kQThreads = 32 * 6;
constexpr int kQABytes = kQM * kQK * 2, kQBBytes = kQN * kQK * 2;          // 16 KB + 32 KB per stage
constexpr int kQOffB = kQStages * kQABytes;
constexpr int kQOffBars = kQOffB + kQStages * kQBBytes;                    // full[4] empty[4] tfull[2] tempty[2]
constexpr int kQOffTmem = kQOffBars + 12 * 8;
constexpr int kQSmemAlloc = kQOffTmem + 16 + 1024;
thread_local char g_q_err[256] = "";

struct QArgs {
  __nv_bfloat16* out;
  const int32_t* positions;       // [T] or nullptr (no rotary embedding)
  const float2* tab_hi;           // [n_hi][d/2] (cos, sin) of (256 p) f_c
  const float2* tab_lo;           // [256][d/2]  (cos, sin) of p f_c
  int n_hi, T, N, Dm, d, Hq, tiles_m, tiles_n;
};

__global__ void rope_tables_kernel(double theta, int d, int n_hi, float2* tab_hi, float2* tab_lo) {
  const int half = d / 2;
  const int total = (n_hi + 256) * half;
  for (int x = blockIdx.x * blockDim.x + threadIdx.x; x < total; x += gridDim.x * blockDim.x) {
    const int p = x / half, c = x % half;
    const double f = pow(theta, -2.0 * (double)c / (double)d);
    const double a = (p < n_hi ? 256.0 * (double)p : (double)(p - n_hi)) * f;
    const float2 v = make_float2((float)cos(a), (float)sin(a));
    if (p < n_hi) tab_hi[(size_t)p * half + c] = v; else tab_lo[(size_t)(p - n_hi) * half + c] = v;
  }
}

__device__ __forceinline__ void tmem_ld_32x32b_x8(uint32_t taddr, uint32_t* r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr) : "memory");
}
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

__global__ void __launch_bounds__(kQThreads, 1)
qproj_kernel(const __grid_constant__ CUtensorMap a_map, const __grid_constant__ CUtensorMap b_map, const QArgs q) {
  extern __shared__ unsigned char smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* gbase = smem_raw + (base - raw);
  const uint32_t sA = base, sB = base + kQOffB, bars = base + kQOffBars;
  const uint32_t full = bars, empty = bars + 32, tfull = bars + 64, tempty = bars + 80;
  volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(gbase + kQOffTmem);
  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int i = 0; i < kQStages; ++i) { mbar_init(full + 8 * i, 1); mbar_init(empty + 8 * i, 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(tfull + 8 * i, 1); mbar_init(tempty + 8 * i, 4); }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(smem_u32((const void*)tmem_ptr), 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_ptr;
  const int n_tiles = q.tiles_m * q.tiles_n, k_steps = q.Dm / kQK;

  if (warp == 0) {
    // ================================ TMA producer ================================
    if (lane == 0) {
      int it = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int m0 = (tile / q.tiles_n) * kQM, n0 = (tile % q.tiles_n) * kQN;
        for (int ks = 0; ks < k_steps; ++ks, ++it) {
          const int st = it % kQStages, use = it / kQStages;
          mbar_wait_backoff(empty + 8 * st, (use & 1) ^ 1);
          mbar_expect_tx(full + 8 * st, kQABytes + kQBBytes);
          tma_load_2d(sA + st * kQABytes, &a_map, full + 8 * st, ks * kQK, m0);
          tma_load_2d(sB + st * kQBBytes, &b_map, full + 8 * st, ks * kQK, n0);
        }
      }
    }
  } else if (warp == 1) {
    // ================================ MMA issuer ================================
    constexpr uint32_t kDescHi = (uint32_t)(1024u >> 4) | (1u << 14) | (2u << 29);   // SBO | version | SWIZZLE_128B
    constexpr uint32_t kDescLo = 1u << 16;
    const uint32_t idesc = make_idesc_bf16(kQN);
    int it = 0, tile_iter = 0;
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++tile_iter) {
      const int buf = tile_iter & 1, tuse = tile_iter >> 1;
      mbar_wait(tempty + 8 * buf, (tuse & 1) ^ 1);
      tc_fence_after();
      const uint32_t d_tmem = tmem_base + buf * kQN;
      for (int ks = 0; ks < k_steps; ++ks, ++it) {
        const int st = it % kQStages, use = it / kQStages;
        mbar_wait(full + 8 * st, use & 1);
        tc_fence_after();
        if (elect_one()) {
          const uint32_t a_lo = ((sA + st * kQABytes) >> 4) | kDescLo, b_lo = ((sB + st * kQBBytes) >> 4) | kDescLo;
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const uint64_t ad = ((uint64_t)kDescHi << 32) | (a_lo + ((k * 32) >> 4));
            const uint64_t bd = ((uint64_t)kDescHi << 32) | (b_lo + ((k * 32) >> 4));
            umma_bf16(d_tmem, ad, bd, idesc, (ks | k) != 0);
          }
          umma_commit(empty + 8 * st);                         // the stage is free once these MMAs have read it
          if (ks == k_steps - 1) umma_commit(tfull + 8 * buf);   // accumulator complete
        }
        __syncwarp();
      }
    }
  } else {
    // ================================ epilogue: RoPE + bf16 + layout ================================
    const int quad = warp & 3;                                  // TMEM lane quadrant of this warp
    const int half = q.d / 2, heads_per_tile = kQN / q.d;
    int tile_iter = 0;
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++tile_iter) {
      const int buf = tile_iter & 1, tuse = tile_iter >> 1;
      const int m0 = (tile / q.tiles_n) * kQM, n0 = (tile % q.tiles_n) * kQN;
      const int row = m0 + quad * 32 + lane;
      const bool row_ok = row < q.T;
      int pos = 0;
      if (q.positions && row_ok) pos = q.positions[row];
      const float2* th = q.tab_hi + (size_t)min(max(pos >> 8, 0), q.n_hi - 1) * half;
      const float2* tl = q.tab_lo + (size_t)(pos & 255) * half;
      mbar_wait(tfull + 8 * buf, tuse & 1);
      tc_fence_after();
      const uint32_t ta = tmem_base + ((uint32_t)(quad * 32) << 16) + buf * kQN;
      for (int hh = 0; hh < heads_per_tile; ++hh) {
        const int head = n0 / q.d + hh;
        if (head >= q.Hq) break;                               // (warp-uniform)
        __nv_bfloat16* o = q.out + ((size_t)row * q.Hq + head) * q.d;
        for (int c0 = 0; c0 < half; c0 += 16) {
          uint32_t lo[16], hi[16];
          tmem_ld_32x32b_x8(ta + hh * q.d + c0, lo);
          tmem_ld_32x32b_x8(ta + hh * q.d + c0 + 8, lo + 8);
          tmem_ld_32x32b_x8(ta + hh * q.d + half + c0, hi);
          tmem_ld_32x32b_x8(ta + hh * q.d + half + c0 + 8, hi + 8);
          tmem_wait_ld();
          float x[16], y[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) { x[i] = __uint_as_float(lo[i]); y[i] = __uint_as_float(hi[i]); }
          if (q.positions) {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
              const float2 a = th[c0 + i], b = tl[c0 + i];
              const float cs = a.x * b.x - a.y * b.y, sn = a.y * b.x + a.x * b.y;   // cos / sin of the summed angle
              const float xr = x[i] * cs - y[i] * sn, yr = y[i] * cs + x[i] * sn;
              x[i] = xr; y[i] = yr;
            }
          }
          if (row_ok) {
            uint4 v0 = make_uint4(pack_bf16x2(x[0], x[1]), pack_bf16x2(x[2], x[3]), pack_bf16x2(x[4], x[5]), pack_bf16x2(x[6], x[7]));
            uint4 v1 = make_uint4(pack_bf16x2(x[8], x[9]), pack_bf16x2(x[10], x[11]), pack_bf16x2(x[12], x[13]), pack_bf16x2(x[14], x[15]));
            uint4 w0 = make_uint4(pack_bf16x2(y[0], y[1]), pack_bf16x2(y[2], y[3]), pack_bf16x2(y[4], y[5]), pack_bf16x2(y[6], y[7]));
            uint4 w1 = make_uint4(pack_bf16x2(y[8], y[9]), pack_bf16x2(y[10], y[11]), pack_bf16x2(y[12], y[13]), pack_bf16x2(y[14], y[15]));
            *reinterpret_cast<uint4*>(o + c0) = v0;
            *reinterpret_cast<uint4*>(o + c0 + 8) = v1;
            *reinterpret_cast<uint4*>(o + half + c0) = w0;
            *reinterpret_cast<uint4*>(o + half + c0 + 8) = w1;
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty + 8 * buf);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) { tc_fence_after(); tmem_dealloc(tmem_base, 512); }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn q_get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult r;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &r) == cudaSuccess &&
        r == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}
int q_fail(int code, const char* msg) { snprintf(g_q_err, sizeof g_q_err, "%s", msg); return code; }

}  // namespace

const char* qproj_error() { return g_q_err; }

size_t qproj_workspace_bytes(int max_position, int d) {
  if (max_position < 0 || d <= 0) return 0;
  return sizeof(float2) * (size_t)((max_position >> 8) + 1 + 256) * (d / 2);
}

int qproj_launch(const void* hidden, const void* wq, const int32_t* positions, int max_position, double theta, int T,
                 int Dm, int Hq, int d, void* out, void* workspace, size_t workspace_bytes, cudaStream_t st) {
  if (T == 0) return KARA_OK;
  int dev = 0, cc_major = 0, num_sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return q_fail(KARA_ECUDA, "no CUDA device");
  if (cc_major != 10) return q_fail(KARA_EUNSUPPORTED, "the window-query producer needs an sm_100 device");
  EncodeTiledFn enc = q_get_encode();
  if (!enc) return q_fail(KARA_ECUDA, "cuTensorMapEncodeTiled entry point not found");
  const int N = Hq * d;
  const int n_hi = (max_position >> 8) + 1;
  float2* tab_hi = static_cast<float2*>(workspace);
  float2* tab_lo = tab_hi + (size_t)n_hi * (d / 2);
  if (positions) {
    if (workspace_bytes < qproj_workspace_bytes(max_position, d)) return q_fail(KARA_ENOMEM, "workspace too small for the rotary tables");
    rope_tables_kernel<<<64, 256, 0, st>>>(theta, d, n_hi, tab_hi, tab_lo);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return q_fail(KARA_ECUDA, cudaGetErrorString(e));
  }
  CUtensorMap amap, bmap;
  cuuint32_t estr[2] = {1u, 1u};
  {
    cuuint64_t dims[2] = {(cuuint64_t)Dm, (cuuint64_t)T};
    cuuint64_t strides[1] = {(cuuint64_t)Dm * 2};
    cuuint32_t box[2] = {(cuuint32_t)kQK, (cuuint32_t)kQM};
    if (enc(&amap, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(hidden), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return q_fail(KARA_ECUDA, "cuTensorMapEncodeTiled(hidden) failed");
  }
  {
    cuuint64_t dims[2] = {(cuuint64_t)Dm, (cuuint64_t)N};
    cuuint64_t strides[1] = {(cuuint64_t)Dm * 2};
    cuuint32_t box[2] = {(cuuint32_t)kQK, (cuuint32_t)kQN};
    if (enc(&bmap, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(wq), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return q_fail(KARA_ECUDA, "cuTensorMapEncodeTiled(wq) failed");
  }
  QArgs q{static_cast<__nv_bfloat16*>(out), positions, tab_hi, tab_lo, n_hi, T, N, Dm, d, Hq,
          (T + kQM - 1) / kQM, (N + kQN - 1) / kQN};
  if (cudaFuncSetAttribute(qproj_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kQSmemAlloc) != cudaSuccess)
    return q_fail(KARA_ECUDA, "cudaFuncSetAttribute(max dynamic smem) failed");
  const int n_tiles = q.tiles_m * q.tiles_n;
  const int grid = n_tiles < num_sms ? n_tiles : num_sms;
  qproj_kernel<<<grid, kQThreads, kQSmemAlloc, st>>>(amap, bmap, q);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return q_fail(KARA_ECUDA, cudaGetErrorString(e));
  return KARA_OK;
}

}  // namespace kara
