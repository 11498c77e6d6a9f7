// score_simt.cu — a1 (Eq. 4) on CUDA cores: the simple, shape-agnostic score
// kernel.  It is the debug cross-check of the tcgen05 path (KARA_SCORE_SIMT) and the path for
// shapes that kernel does not take.  fp32 accumulation; deterministic summation order.
//
// grid = (units, parts).  A CTA owns a contiguous range of the unit's query rows
// r = (i - q_row_begin)*G + g; a warp owns one row at a time: lanes split the keys, the row's
// logits live in a warp-private smem strip, softmax by warp shuffles, and p is accumulated into
// a warp-private column strip (lane owns columns j = lane mod 32: no conflicts, fixed order).
// The 8 warp strips are summed in warp order into partial[unit][part][:].
#include "kara_internal.h"

namespace kara {

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__global__ void __launch_bounds__(kThreads) score_simt_kernel(const Call c) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = c.n, n_pad = c.n_pad, d = c.g.d;
  float* s_logit = reinterpret_cast<float*>(smem_raw);          // [kWarps][n_pad]
  float* s_acc = s_logit + kWarps * n_pad;                      // [kWarps][n_pad]
  float* s_q = s_acc + kWarps * n_pad;                          // [kWarps][d]
  long long* s_koff = reinterpret_cast<long long*>(s_q + kWarps * d);  // [n_pad] key row offsets

  const int unit = blockIdx.x, part = blockIdx.y;
  int li, s, w, hk;
  unit_decode(unit, c.n_seqs, c.n_windows, c.g.n_kv_heads, li, s, w, hk);
  const int layer = c.layer_begin + li;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float* out = c.partial + ((long long)unit * c.parts + part) * n_pad;

  int h, t, len;
  const bool ok = window_of(c, s, h, t, len);
  h += w * c.W;                                            // this unit's window
  for (int j = threadIdx.x; j < n; j += kThreads) s_koff[j] = ok ? row_offset(c, layer, s, hk, h + j) : -1;
  for (int j = threadIdx.x; j < kWarps * n_pad; j += kThreads) s_acc[j] = 0.f;
  __syncthreads();
  bool bad = !ok;
  for (int j = threadIdx.x; j < n; j += kThreads) bad |= (s_koff[j] < 0);
  if (__syncthreads_or(bad)) {   // skipped unit: zero scores (status word already says why)
    for (int j = threadIdx.x; j < n_pad; j += kThreads) out[j] = 0.f;
    return;
  }

  const int rows = (c.W - c.q_row_begin) * c.G;
  const int rows_per_part = (rows + c.parts - 1) / c.parts;
  const int r0 = part * rows_per_part;
  const int r1 = min(rows, r0 + rows_per_part);
  const float scale = rsqrtf((float)d);
  float* my_logit = s_logit + warp * n_pad;
  float* my_acc = s_acc + warp * n_pad;
  float* my_q = s_q + warp * d;

  for (int r = r0 + warp; r < r1; r += kWarps) {
    const int i = c.q_row_begin + r / c.G, g = r % c.G;
    const __nv_bfloat16* q = c.window_q +
        (((((long long)li * c.n_seqs + s) * c.n_windows + w) * c.W + i) * c.n_q_heads + (hk * c.G + g)) * (long long)d;
    for (int x = lane; x < d; x += 32) my_q[x] = __bfloat162float(q[x]);
    __syncwarp();
    float m = -INFINITY;
    for (int j = lane; j < n; j += 32) {
      const uint4* kr = reinterpret_cast<const uint4*>(c.k_pool + s_koff[j]);
      float acc = 0.f;
      for (int v = 0; v < d / 8; ++v) {
        const uint4 pk = __ldg(kr + v);
        const __nv_bfloat162* h2 = reinterpret_cast<const __nv_bfloat162*>(&pk);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float2 f = __bfloat1622float2(h2[e]);
          acc = fmaf(my_q[v * 8 + 2 * e], f.x, acc);
          acc = fmaf(my_q[v * 8 + 2 * e + 1], f.y, acc);
        }
      }
      const float sj = acc * scale;
      my_logit[j] = sj;
      m = fmaxf(m, sj);
    }
    m = warp_max(m);
    float l = 0.f;
    for (int j = lane; j < n; j += 32) {
      const float e = __expf(my_logit[j] - m);
      my_logit[j] = e;
      l += e;
    }
    l = warp_sum(l);
    const float inv = 1.f / l;
    for (int j = lane; j < n; j += 32) my_acc[j] += my_logit[j] * inv;
    __syncwarp();
  }
  __syncthreads();
  for (int j = threadIdx.x; j < n_pad; j += kThreads) {
    float a = 0.f;
    if (j < n)
#pragma unroll
      for (int w = 0; w < kWarps; ++w) a += s_acc[w * n_pad + j];
    out[j] = a;
  }
}

}  // namespace

cudaError_t launch_score_simt(const Call& c, cudaStream_t st) {
  const int units = unit_count(c);
  const size_t smem = sizeof(float) * (size_t)(2 * kWarps * c.n_pad + kWarps * c.g.d) +
                      sizeof(long long) * (size_t)c.n_pad;
  cudaError_t e = cudaFuncSetAttribute(score_simt_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  score_simt_kernel<<<dim3(units, c.parts), kThreads, smem, st>>>(c);
  return cudaGetLastError();
}

}  // namespace kara
