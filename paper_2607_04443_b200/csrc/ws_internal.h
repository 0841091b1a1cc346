// Internal helpers shared by the ws_*.cu translation units (NOT part of the C ABI, and not
// shared with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ws.h"

namespace wsi {

// Records a CUDA error for ws_last_cuda_error() and returns WS_ERR_CUDA.
int cuda_fail(cudaError_t e);
// Bumps the process-wide launch counter reported by ws_kernel_launch_count().
void count_launch(int n = 1);

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline bool aligned256(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 255u) == 0; }
inline int elem_bytes(ws_dtype dt) { return dt == WS_DTYPE_BF16 ? 2 : (dt == WS_DTYPE_F32 ? 4 : 0); }
inline bool ranges_overlap(const void* a, size_t na, const void* b, size_t nb) {
  const uintptr_t a0 = reinterpret_cast<uintptr_t>(a), b0 = reinterpret_cast<uintptr_t>(b);
  return na != 0 && nb != 0 && a0 < b0 + nb && b0 < a0 + na;
}

// Host-only argument checks of ws_block_causal_attn (ws_attn.cu) and ws_kv_cache_write (ws_copy.cu): no device is
// touched and nothing is launched, so a composite entry point can run them before it enqueues anything.
int attn_validate(const void* out, const float* lse, const void* q, const void* k_cache, const void* v_cache, int64_t capacity,
                  int64_t cache_len, const void* k_new, const void* v_new, int32_t Ln, int32_t H, int32_t d, int32_t Lq,
                  const ws_block_mask* mask, float softmax_scale, const void* workspace, size_t workspace_bytes, ws_dtype dt);
// ws_block_causal_attn on BF16 inputs with the output rows written as FP32 [Lq, H, d] (ws_attn.cu; used by ws_unit.cu
// for partial results that are merged afterwards).  Arguments and errors as ws_block_causal_attn with WS_DTYPE_BF16.
int attn_bf16_in_f32_out(float* out, float* lse, const void* q, const void* k_cache, const void* v_cache, int64_t capacity,
                         int64_t cache_len, const void* k_new, const void* v_new, int32_t Ln, int32_t H, int32_t d, int32_t Lq,
                         const ws_block_mask* mask, float softmax_scale, void* workspace, size_t workspace_bytes, void* stream);
int cache_write_validate(const void* k_cache, const void* v_cache, int64_t capacity, int32_t H, int32_t d, const void* k_src,
                         const void* v_src, int32_t n_rows, int32_t H_src, int32_t head_begin, int64_t row_offset, ws_dtype dt);

// After a launch: pick up launch-configuration errors without synchronising.
inline int after_launch(int n_launches) {
  cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) {
    (void)cudaGetLastError();
    return cuda_fail(e);
  }
  count_launch(n_launches);
  return WS_OK;
}

// ---- programmatic dependent launch (PDL) ----
// The hot path is a chain of short kernels on one stream (cache write, relayouts, attention, relayout); the
// kernel-to-kernel gap is of the order of a relayout's whole HBM time.  Every kernel of the library is launched
// with programmatic stream serialisation: its CTAs may be scheduled while the previous kernel drains, run their
// address set-up, and block in pdl_wait() -- which returns once the previous kernel has completed and its
// writes are visible -- before their FIRST global-memory access.  pdl_trigger() lets the next kernel do the same.
// A successor that is not one of ours (no attribute) is serialised as usual.  Capturable in CUDA graphs.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
#endif

}  // namespace wsi
