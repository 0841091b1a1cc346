// ws_unit.cu -- ws_unit_forward_host: one streaming unit end to end from HOST buffers
// (include/ws.h a5).  Orchestration of the library's own kernels around plain cudaMemcpyAsync calls:
//
//   copy-in stream :  K/V slice  |  Q[0]  |  K_new[0], V_new[0]  |  Q[1]  |  K_new[1], V_new[1]  | ...
//   caller's stream:  cache write -> A[0]: attention of Q[0] against the CACHE  (while K_new / V_new are still in flight)
//                                 -> B[0]: attention of Q[0] against the unit's own rows -> LSE-weighted merge of A and B
//   copy-out stream:                                                                        out[0] -> host  | ...
//
// Every transfer is ONE contiguous copy (measured on the B200 host, PCIe Gen5 x16: 55 GB/s, against 30-44 GB/s for
// cudaMemcpy2DAsync of any row width), and the big part of the attention -- the cached keys, 94 % of them at config 3
// -- runs under the transfer of the unit's own K/V.  What follows the last input byte is B (970 keys), the merge and the
// output copy.  The merge is the split-KV identity the oracle pins (attention over A u B = LSE-weighted mean of attention
// over A and over B); nothing is computed on the host.
#include <cuda_bf16.h>

#include <mutex>

#include "ws_internal.h"

namespace {
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Staging {
  size_t k_slice, v_slice, q, k_new, v_new, out, out_a, out_b, lse_a, lse_b, attn_ws, attn_ws_bytes, total;
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
  s.out_a = off; off = align_up(off + (size_t)Lq * H * d * 4, 256);  // the two partial results stay FP32 until they are merged
  s.out_b = off; off = align_up(off + (size_t)Lq * H * d * 4, 256);
  s.lse_a = off; off = align_up(off + (size_t)Lq * H * 4, 256);
  s.lse_b = off; off = align_up(off + (size_t)Lq * H * 4, 256);
  s.attn_ws = off;
  s.attn_ws_bytes = ws_block_causal_attn_workspace_bytes(Lq, H, d, kv_total, WS_DTYPE_BF16);
  off = align_up(off + s.attn_ws_bytes, 256);
  s.total = off;
  return s;
}

// out[i, h, :] = (w_a O_a[i, h, :] + w_b O_b[i, h, :]),  w_x = exp(lse_x[h, i] - logaddexp(lse_a, lse_b)[h, i]):
// attention over the union of two disjoint key sets from the attention over each (natural-log LSE, [H, Lq]).
// O_a, O_b are FP32 (the partial attentions' normalised rows before any rounding), so the merged row is rounded to
// BF16 exactly once, like ws_block_causal_attn's.  One thread per 8 elements (two 16-byte loads per side, one 16-byte
// store).  A side whose LSE is -inf saw no key and gets weight 0.
__global__ void __launch_bounds__(256) merge_two_kernel(uint4* __restrict__ out, const float4* __restrict__ oa, const float4* __restrict__ ob,
                                                        const float* __restrict__ lse_a, const float* __restrict__ lse_b, int32_t Lq,
                                                        int32_t H, int32_t d8) {
  wsi::pdl_trigger();
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, total = (int64_t)Lq * H * d8;
  wsi::pdl_wait();
  if (idx >= total) return;
  const int64_t ih = idx / d8;
  const int i = (int)(ih / H), h = (int)(ih - (int64_t)i * H);
  const float la = lse_a[(int64_t)h * Lq + i], lb = lse_b[(int64_t)h * Lq + i];
  const float m = fmaxf(la, lb);
  float wa = 0.f, wb = 0.f;
  if (m > -INFINITY) {
    const float ea = __expf(la - m), eb = __expf(lb - m), inv = 1.f / (ea + eb);
    wa = ea * inv;
    wb = eb * inv;
  }
  const float4 a0 = oa[2 * idx], a1 = oa[2 * idx + 1], b0 = ob[2 * idx], b1 = ob[2 * idx + 1];
  auto pack = [wa, wb](float ax, float bx, float ay, float by) {
    const __nv_bfloat162 p = __floats2bfloat162_rn(wa * ax + wb * bx, wa * ay + wb * by);
    return *reinterpret_cast<const uint32_t*>(&p);
  };
  out[idx] = make_uint4(pack(a0.x, b0.x, a0.y, b0.y), pack(a0.z, b0.z, a0.w, b0.w), pack(a1.x, b1.x, a1.y, b1.y),
                        pack(a1.z, b1.z, a1.w, b1.w));
}

// Internal helper streams and events of ws_unit_forward_host (one set per device, created on first use).
struct Pipe {
  cudaStream_t copy_in = nullptr, copy_out = nullptr;
  cudaEvent_t fork = nullptr, join = nullptr, join_out = nullptr, in_ready = nullptr, out_ready = nullptr;
  std::mutex enqueue_mu;  // held while a call enqueues its work: the events above are shared by all calls on the device
};
Pipe* get_pipe() {
  static std::mutex mu;
  static Pipe pipes[64];
  static bool ready[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
  std::lock_guard<std::mutex> lock(mu);
  if (!ready[dev]) {
    Pipe& p = pipes[dev];
    const bool ok = cudaStreamCreateWithFlags(&p.copy_in, cudaStreamNonBlocking) == cudaSuccess &&
                    cudaStreamCreateWithFlags(&p.copy_out, cudaStreamNonBlocking) == cudaSuccess &&
                    cudaEventCreateWithFlags(&p.fork, cudaEventDisableTiming) == cudaSuccess &&
                    cudaEventCreateWithFlags(&p.join, cudaEventDisableTiming) == cudaSuccess &&
                    cudaEventCreateWithFlags(&p.join_out, cudaEventDisableTiming) == cudaSuccess &&
                    cudaEventCreateWithFlags(&p.in_ready, cudaEventDisableTiming) == cudaSuccess &&
                    cudaEventCreateWithFlags(&p.out_ready, cudaEventDisableTiming) == cudaSuccess;
    if (!ok) return nullptr;
    ready[dev] = true;
  }
  return &pipes[dev];
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
  // ---- every check of this call and of the calls it is made of, before anything is enqueued ----
  if (!out_host || !q_host || !k_cache || !v_cache || Lq <= 0 || Ln < 0 || n_steps <= 0 || H <= 0 || n_slice_rows < 0)
    return WS_ERR_INVALID_ARG;
  if ((Ln > 0) != (k_new_host != nullptr) || (Ln > 0) != (v_new_host != nullptr)) return WS_ERR_INVALID_ARG;
  if ((n_slice_rows > 0) != (k_slice_host != nullptr) || (n_slice_rows > 0) != (v_slice_host != nullptr)) return WS_ERR_INVALID_ARG;
  if (d != 64 && d != 128) return WS_ERR_UNSUPPORTED;
  if (capacity <= 0 || row_offset < 0 || row_offset + n_slice_rows > capacity || cache_len_after < 0 || cache_len_after > capacity)
    return WS_ERR_OUT_OF_RANGE;
  if (cache_len_after + Ln > 0x7fffffffLL - 128) return WS_ERR_UNSUPPORTED;
  const Staging s = staging_layout(Lq, Ln, H, d, n_slice_rows, cache_len_after + Ln, n_steps);
  if (!staging || staging_bytes < s.total || !wsi::aligned256(staging)) return WS_ERR_WORKSPACE;
  char* st = reinterpret_cast<char*>(staging);
  const size_t step_q = (size_t)Lq * H * d * 2, step_n = (size_t)Ln * H * d * 2, slice_b = (size_t)n_slice_rows * H * d * 2;
  const bool has_cache = cache_len_after > 0, has_new = Ln > 0, both = has_cache && has_new;
  const int32_t q_end = Lq, vis_a = (int32_t)cache_len_after, vis_b = Ln, vis_none = 0;
  const ws_block_mask mask_a{1, &q_end, &vis_a}, mask_b{1, &q_end, &vis_b}, mask_none{1, &q_end, &vis_none};
  float* lse_a = reinterpret_cast<float*>(st + s.lse_a);
  float* lse_b = reinterpret_cast<float*>(st + s.lse_b);
  if (n_slice_rows > 0)
    if (const int rc = wsi::cache_write_validate(k_cache, v_cache, capacity, H, d, st + s.k_slice, st + s.v_slice, n_slice_rows, H, 0,
                                                 row_offset, WS_DTYPE_BF16))
      return rc;
  if (has_cache || !has_new)
    if (const int rc = wsi::attn_validate(st + s.out_a, lse_a, st + s.q, k_cache, v_cache, capacity, cache_len_after, nullptr, nullptr, 0, H, d,
                                          Lq, has_cache ? &mask_a : &mask_none, softmax_scale, st + s.attn_ws, s.attn_ws_bytes, WS_DTYPE_BF16))
      return rc;
  if (has_new)
    if (const int rc = wsi::attn_validate(st + s.out_b, lse_b, st + s.q, k_cache, v_cache, capacity, 0, st + s.k_new, st + s.v_new, Ln, H, d, Lq,
                                          &mask_b, softmax_scale, st + s.attn_ws, s.attn_ws_bytes, WS_DTYPE_BF16))
      return rc;

  Pipe* pipe = get_pipe();
  if (!pipe) return wsi::cuda_fail(cudaErrorUnknown);
  // One set of events per device: calls on the same device are serialised on the host for the length of the enqueue.
  std::lock_guard<std::mutex> enqueue_lock(pipe->enqueue_mu);
  cudaError_t e = cudaEventRecord(pipe->fork, stream);
  if (e != cudaSuccess) return wsi::cuda_fail(e);  // nothing has been forked yet
  int rc = WS_OK;
  e = cudaStreamWaitEvent(pipe->copy_in, pipe->fork, 0);
  const bool in_forked = e == cudaSuccess;
  if (e == cudaSuccess) e = cudaStreamWaitEvent(pipe->copy_out, pipe->fork, 0);
  const bool out_forked = in_forked && e == cudaSuccess;
  auto h2d = [&](size_t dst_off, const void* src, size_t bytes) {
    if (e == cudaSuccess && bytes > 0) e = cudaMemcpyAsync(st + dst_off, src, bytes, cudaMemcpyHostToDevice, pipe->copy_in);
  };
  // the helper stream's progress so far becomes a dependency of the caller's stream (the event is re-recorded per use:
  // a wait refers to the record that preceded it)
  auto inputs_arrived = [&]() {
    if (e == cudaSuccess) e = cudaEventRecord(pipe->in_ready, pipe->copy_in);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, pipe->in_ready, 0);
  };
  // ---- the slice and the cache write ----
  if (n_slice_rows > 0) {
    h2d(s.k_slice, k_slice_host, slice_b);
    h2d(s.v_slice, v_slice_host, slice_b);
    inputs_arrived();
    if (e == cudaSuccess)
      rc = ws_kv_cache_write(k_cache, v_cache, capacity, H, d, st + s.k_slice, st + s.v_slice, n_slice_rows, H, 0, row_offset, WS_DTYPE_BF16,
                             stream);
  }
  // ---- the denoising steps ----
  for (int32_t step = 0; step < n_steps && e == cudaSuccess && rc == WS_OK; ++step) {
    char* q_s = st + s.q + step * step_q;
    char* out_s = st + s.out + step * step_q;
    h2d(s.q + step * step_q, static_cast<const char*>(q_host) + step * step_q, step_q);
    inputs_arrived();
    if (e != cudaSuccess) break;
    if (both)  // A: the cached keys, as an FP32 partial result
      rc = wsi::attn_bf16_in_f32_out(reinterpret_cast<float*>(st + s.out_a), lse_a, q_s, k_cache, v_cache, capacity, cache_len_after, nullptr,
                                     nullptr, 0, H, d, Lq, &mask_a, softmax_scale, st + s.attn_ws, s.attn_ws_bytes, stream);
    else if (has_cache || !has_new)  // the cached keys are all there is (or, with no key at all, the zero / -inf result)
      rc = ws_block_causal_attn(out_s, nullptr, q_s, k_cache, v_cache, capacity, cache_len_after, nullptr, nullptr, 0, H, d, Lq,
                                has_cache ? &mask_a : &mask_none, softmax_scale, st + s.attn_ws, s.attn_ws_bytes, WS_DTYPE_BF16, stream);
    if (has_new && rc == WS_OK) {
      h2d(s.k_new + step * step_n, static_cast<const char*>(k_new_host) + step * step_n, step_n);
      h2d(s.v_new + step * step_n, static_cast<const char*>(v_new_host) + step * step_n, step_n);
      inputs_arrived();
      if (e != cudaSuccess) break;
      // B: the unit's own rows
      if (both)
        rc = wsi::attn_bf16_in_f32_out(reinterpret_cast<float*>(st + s.out_b), lse_b, q_s, k_cache, v_cache, capacity, 0,
                                       st + s.k_new + step * step_n, st + s.v_new + step * step_n, Ln, H, d, Lq, &mask_b, softmax_scale,
                                       st + s.attn_ws, s.attn_ws_bytes, stream);
      else
        rc = ws_block_causal_attn(out_s, nullptr, q_s, k_cache, v_cache, capacity, 0, st + s.k_new + step * step_n,
                                  st + s.v_new + step * step_n, Ln, H, d, Lq, &mask_b, softmax_scale, st + s.attn_ws, s.attn_ws_bytes,
                                  WS_DTYPE_BF16, stream);
      if (both && rc == WS_OK) {
        const int64_t total = (int64_t)Lq * H * (d / 8);
        e = wsi::launch_pdl(merge_two_kernel, dim3((unsigned)((total + 255) / 256)), dim3(256), 0, stream, reinterpret_cast<uint4*>(out_s),
                            reinterpret_cast<const float4*>(st + s.out_a), reinterpret_cast<const float4*>(st + s.out_b),
                            (const float*)lse_a, (const float*)lse_b, Lq, H, d / 8);
        if (e == cudaSuccess) wsi::count_launch(1);
      }
    }
    if (rc != WS_OK || e != cudaSuccess) break;
    e = cudaEventRecord(pipe->out_ready, stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(pipe->copy_out, pipe->out_ready, 0);
    if (e == cudaSuccess)
      e = cudaMemcpyAsync(static_cast<char*>(out_host) + step * step_q, out_s, step_q, cudaMemcpyDeviceToHost, pipe->copy_out);
  }
  // ---- join both helper streams back into `stream`, whatever happened above ----
  cudaError_t je = cudaSuccess;
  if (in_forked) {
    je = cudaEventRecord(pipe->join, pipe->copy_in);
    if (je == cudaSuccess) je = cudaStreamWaitEvent(stream, pipe->join, 0);
  }
  if (out_forked) {
    cudaError_t je2 = cudaEventRecord(pipe->join_out, pipe->copy_out);
    if (je2 == cudaSuccess) je2 = cudaStreamWaitEvent(stream, pipe->join_out, 0);
    if (je == cudaSuccess) je = je2;
  }
  if (rc != WS_OK) return rc;
  if (e != cudaSuccess) return wsi::cuda_fail(e);
  if (je != cudaSuccess) return wsi::cuda_fail(je);
  return WS_OK;
}
