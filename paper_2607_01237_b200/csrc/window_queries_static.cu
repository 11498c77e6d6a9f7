// window_queries_static.cu — kara_window_queries_static (include/kara.h): the window-query producer for callers that may
// not allocate device memory and have no workspace to lend (a serving engine in the middle of decoding: its HBM is all
// in the KV pool, a cudaMalloc there fails or stalls the device, and its allocator policy forbids one anyway).
//
// The only scratch the producer needs are the rotary cos / sin tables (qproj.cu: tab_hi / tab_lo).  Here they live in
// g_kara_static_scratch below, which is part of this library's device image: no cudaMalloc, no cudaFree, no allocating
// library routine on this path, at the cost of KARA_STATIC_SCRATCH_BYTES of HBM on every GPU that loads the library.
//
// In host code the NAME of a __device__ array is only a handle for the runtime, not a pointer a kernel can use, so the
// array's real address is asked for once per device (cudaGetSymbolAddress, with that device current) and that address is
// what travels to the kernels.  The array has internal linkage, which is why the lookup has to live in this file.
#include <mutex>

#include "kara_internal.h"

// One per GPU; rewritten by every call (see "Sharing" in include/kara.h).  256-byte alignment is what the ABI asks of a workspace.
static __device__ __align__(256) unsigned char g_kara_static_scratch[KARA_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_addr_mutex;
void* g_scratch_addr[kMaxDevices] = {};   // device address of g_kara_static_scratch on device i; nullptr = not looked up yet

// The address of the array on the CURRENT device: looked up on the first call per device, then served from the table.
int scratch_of_current_device(void** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return kara::api_fail(KARA_ECUDA, "kara_window_queries_static: cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxDevices)
    return kara::api_fail(KARA_EUNSUPPORTED, "kara_window_queries_static: device ordinal %d outside [0,%d)", dev, kMaxDevices);
  std::lock_guard<std::mutex> lock(g_addr_mutex);
  if (!g_scratch_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_kara_static_scratch);
    if (e != cudaSuccess || !p)
      return kara::api_fail(KARA_ECUDA, "kara_window_queries_static: cudaGetSymbolAddress on device %d: %s", dev,
                            cudaGetErrorString(e));
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return KARA_OK;
}

}  // namespace

extern "C" int kara_window_queries_static(const void* hidden, const void* wq, const int32_t* positions, int max_position,
                                          double rope_theta, int n_tokens, int d_model, int n_q_heads, int head_dim,
                                          void* window_q_out, void* stream) {
  // Too many positions for the built-in tables: refused on the host, before any CUDA call.  (A head_dim the producer does
  // not take gives 0 bytes here and is reported by kara_window_queries below.)
  if (positions && max_position >= 0) {
    const size_t need = kara_window_queries_workspace_bytes(max_position, head_dim);
    if (need > (size_t)KARA_STATIC_SCRATCH_BYTES)
      return kara::api_fail(KARA_ENOMEM,
                            "kara_window_queries_static: the rotary tables for max_position=%d at head_dim=%d take %zu bytes, "
                            "the built-in scratch holds %d (max_position <= %d): call kara_window_queries with a workspace of your own",
                            max_position, head_dim, need, KARA_STATIC_SCRATCH_BYTES,
                            (KARA_STATIC_SCRATCH_BYTES / (4 * head_dim) - 256) * 256 - 1);
  }
  void* scratch = nullptr;
  if (positions) {                                   // without positions no table is built or read
    const int rc = scratch_of_current_device(&scratch);
    if (rc != KARA_OK) return rc;
  }
  // Same argument checks, same table kernel, same GEMM as the workspace variant: only where the tables live differs.
  return kara_window_queries(hidden, wq, positions, max_position, rope_theta, n_tokens, d_model, n_q_heads, head_dim,
                             window_q_out, scratch, scratch ? (size_t)KARA_STATIC_SCRATCH_BYTES : 0, stream);
}
