// ws_unit.cu -- ws_unit_forward_host: one streaming unit end to end from HOST buffers
// (include/ws.h a5).  Pure orchestration on one stream: async H2D copies of the
// unit's inputs, ws_kv_cache_write, n_steps x ws_block_causal_attn, async D2H of the outputs.
// Every data-path step is one of the library's own kernels; nothing is computed on the host.
#include "ws_internal.h"

namespace {
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Staging {
  size_t k_slice, v_slice, q, k_new, v_new, out, attn_ws, attn_ws_bytes, total;
};

Staging staging_layout(int32_t Lq, int32_t Ln, int32_t H, int32_t d, int32_t n_slice_rows, int64_t kv_total, int32_t n_steps) {
  Staging s{};
  const size_t es = 2;
  size_t off = 0;
  s.k_slice = off; off = align_up(off + (size_t)n_slice_rows * H * d * es, 256);
  s.v_slice = off; off = align_up(off + (size_t)n_slice_rows * H * d * es, 256);
  s.q = off; off = align_up(off + (size_t)n_steps * Lq * H * d * es, 256);
  s.k_new = off; off = align_up(off + (size_t)n_steps * Ln * H * d * es, 256);
  s.v_new = off; off = align_up(off + (size_t)n_steps * Ln * H * d * es, 256);
  s.out = off; off = align_up(off + (size_t)n_steps * Lq * H * d * es, 256);
  s.attn_ws = off;
  s.attn_ws_bytes = ws_block_causal_attn_workspace_bytes(Lq, H, d, kv_total, WS_DTYPE_BF16);
  off = align_up(off + s.attn_ws_bytes, 256);
  s.total = off;
  return s;
}
}  // namespace

extern "C" __attribute__((visibility("default"))) size_t ws_unit_forward_host_staging_bytes(int32_t Lq, int32_t Ln, int32_t H, int32_t d, int32_t n_slice_rows,
                                                     int64_t kv_total, int32_t n_steps) {
  if (Lq <= 0 || Ln < 0 || H <= 0 || d <= 0 || n_slice_rows < 0 || kv_total < 0 || n_steps <= 0) return 0;
  return staging_layout(Lq, Ln, H, d, n_slice_rows, kv_total, n_steps).total;
}

extern "C" __attribute__((visibility("default"))) int ws_unit_forward_host(void* out_host, const void* q_host, const void* k_new_host, const void* v_new_host,
                                    int32_t Lq, int32_t Ln, int32_t n_steps, void* k_cache, void* v_cache, int64_t capacity,
                                    const void* k_slice_host, const void* v_slice_host, int32_t n_slice_rows, int64_t row_offset,
                                    int64_t cache_len_after, int32_t H, int32_t d, float softmax_scale, void* staging,
                                    size_t staging_bytes, void* stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (!out_host || !q_host || !k_cache || !v_cache || Lq <= 0 || Ln < 0 || n_steps <= 0 || H <= 0 || n_slice_rows < 0)
    return WS_ERR_INVALID_ARG;
  if ((Ln > 0) != (k_new_host != nullptr) || (Ln > 0) != (v_new_host != nullptr)) return WS_ERR_INVALID_ARG;
  if ((n_slice_rows > 0) != (k_slice_host != nullptr) || (n_slice_rows > 0) != (v_slice_host != nullptr)) return WS_ERR_INVALID_ARG;
  if (d != 64 && d != 128) return WS_ERR_UNSUPPORTED;
  if (row_offset < 0 || row_offset + n_slice_rows > capacity || cache_len_after < 0 || cache_len_after > capacity)
    return WS_ERR_OUT_OF_RANGE;
  if (cache_len_after + Ln > 0x7fffffffLL - 128) return WS_ERR_UNSUPPORTED;
  const Staging s = staging_layout(Lq, Ln, H, d, n_slice_rows, cache_len_after + Ln, n_steps);
  if (!staging || staging_bytes < s.total || !wsi::aligned256(staging)) return WS_ERR_WORKSPACE;
  char* st = reinterpret_cast<char*>(staging);
  const size_t step_q = (size_t)Lq * H * d * 2, step_n = (size_t)Ln * H * d * 2, slice_b = (size_t)n_slice_rows * H * d * 2;

  cudaError_t e = cudaSuccess;
  if (n_slice_rows > 0) {
    e = cudaMemcpyAsync(st + s.k_slice, k_slice_host, slice_b, cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(st + s.v_slice, v_slice_host, slice_b, cudaMemcpyHostToDevice, stream);
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(st + s.q, q_host, step_q * n_steps, cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess && Ln > 0) e = cudaMemcpyAsync(st + s.k_new, k_new_host, step_n * n_steps, cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess && Ln > 0) e = cudaMemcpyAsync(st + s.v_new, v_new_host, step_n * n_steps, cudaMemcpyHostToDevice, stream);
  if (e != cudaSuccess) return wsi::cuda_fail(e);

  if (n_slice_rows > 0) {
    int rc = ws_kv_cache_write(k_cache, v_cache, capacity, H, d, st + s.k_slice, st + s.v_slice, n_slice_rows, H, 0, row_offset,
                               WS_DTYPE_BF16, stream);
    if (rc != WS_OK) return rc;
  }
  const int32_t q_end = Lq, kv_vis = (int32_t)(cache_len_after + Ln);
  ws_block_mask mask{1, &q_end, &kv_vis};
  for (int32_t step = 0; step < n_steps; ++step) {
    int rc = ws_block_causal_attn(st + s.out + step * step_q, nullptr, st + s.q + step * step_q, k_cache, v_cache, capacity,
                                  cache_len_after, Ln ? st + s.k_new + step * step_n : nullptr,
                                  Ln ? st + s.v_new + step * step_n : nullptr, Ln, H, d, Lq, &mask, softmax_scale,
                                  st + s.attn_ws, s.attn_ws_bytes, WS_DTYPE_BF16, stream);
    if (rc != WS_OK) return rc;
  }
  e = cudaMemcpyAsync(out_host, st + s.out, step_q * n_steps, cudaMemcpyDeviceToHost, stream);
  if (e != cudaSuccess) return wsi::cuda_fail(e);
  return WS_OK;
}
