// ws_static.cu -- ws_block_causal_attn_static_ws: block-causal unit attention for callers that cannot allocate.
//
// ws_block_causal_attn needs scratch memory in HBM (the FP32 partial results of work items that are split over several
// CTAs, plus BF16 staging copies when the inputs are FP32) and asks its caller to bring it.  Some callers have no way to
// do that:
//   * a performer process whose serving framework reserved all of HBM for its own pools at start-up: cudaMalloc
//     fails there, and the pool's allocator is not reachable from a C plug-in;
//   * the per-unit real-time loop (one unit every 160 ms): cudaMalloc and cudaFree synchronise the
//     whole device, so an allocation made while earlier units are in flight stalls all of them;
//   * code that runs under a "no allocation after initialisation" rule (long-lived sessions that must not fragment or
//     grow the device heap).
// For them the scratch lives in the array below: part of the library's device image, created by the CUDA driver when it
// loads this module on a GPU and released when the process exits.  The entry point itself calls no cudaMalloc,
// cudaFree or allocating library routine; the caller passes only inputs and outputs.
//
// The cost: WS_STATIC_WORKSPACE_BYTES (64 MiB) of HBM are held on EVERY GPU that loads this module, for the life of the
// process, whether the entry point is used or not.
#include <mutex>

#include "ws_internal.h"

namespace {

// The scratch.  In HOST code this name is only a handle for the runtime's symbol table -- it is NOT the device address,
// and a kernel given `g_static_workspace` from host code would fault (or, on a system where the GPU can reach host
// memory, quietly scribble over host memory instead).  Host code must ask the runtime where the array lives on the
// current device: static_workspace_address() below.  (Device code could name the array directly; none here does, the
// attention kernels receive the address like any other workspace pointer.)
static __device__ __align__(256) unsigned char g_static_workspace[WS_STATIC_WORKSPACE_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_addr[kMaxDevices];  // device address of g_static_workspace on device i; nullptr until the first call there

// One-time set-up per device, with that device current: every device has its own copy of the array at its own address.
cudaError_t static_workspace_address(void** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_addr[dev]) {
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_static_workspace);
    if (e != cudaSuccess) return e;
    if (!ptr || !wsi::aligned256(ptr)) return cudaErrorInvalidSymbol;
    g_addr[dev] = ptr;
  }
  *out = g_addr[dev];
  return cudaSuccess;
}

}  // namespace

// See include/ws.h.  Nothing in the scratch has to start at zero: the attention kernel writes every partial record and
// every staging element before the combine kernel (or the attention kernel itself) reads it, which the parity suite
// checks by filling caller workspaces with NaN.  So the array is not cleared between calls; a call simply finds the
// previous call's bytes and overwrites what it uses.
extern "C" __attribute__((visibility("default"))) int ws_block_causal_attn_static_ws(
    void* out, float* lse, const void* q, const void* k_cache, const void* v_cache, int64_t capacity, int64_t cache_len,
    const void* k_new, const void* v_new, int32_t Ln, int32_t H, int32_t d, int32_t Lq, const ws_block_mask* mask,
    float softmax_scale, ws_dtype dt, void* stream) {
  // Every argument rule of ws_block_causal_attn, and the size limit, on the host first (a stand-in address takes the
  // workspace's place: the checks look at its alignment and at the byte count only).  A problem that needs more scratch
  // than the array holds ends here with WS_ERR_WORKSPACE, before any CUDA call.
  const void* stand_in = reinterpret_cast<const void*>(static_cast<uintptr_t>(256));
  if (const int rc = wsi::attn_validate(out, lse, q, k_cache, v_cache, capacity, cache_len, k_new, v_new, Ln, H, d, Lq, mask,
                                        softmax_scale, stand_in, (size_t)WS_STATIC_WORKSPACE_BYTES, dt))
    return rc;
  void* scratch = nullptr;
  const cudaError_t e = static_workspace_address(&scratch);
  if (e != cudaSuccess) return wsi::cuda_fail(e);
  return ws_block_causal_attn(out, lse, q, k_cache, v_cache, capacity, cache_len, k_new, v_new, Ln, H, d, Lq, mask, softmax_scale,
                              scratch, (size_t)WS_STATIC_WORKSPACE_BYTES, dt, stream);
}
