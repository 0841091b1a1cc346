// ws_unit.cu -- ws_unit_forward_host: one streaming unit end to end from HOST buffers
// (include/ws.h a5).  Pure orchestration: async H2D copies of the unit's inputs,
// ws_kv_cache_write, n_steps x attention, async D2H of the outputs, pipelined over four head groups
// so that the PCIe transfers in both directions overlap the kernels.  Every data-path step is one
// of the library's own kernels; nothing is computed on the host.
#include <mutex>

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

// Internal helper streams and events of ws_unit_forward_host (one set per device, created on first use).
constexpr int kGroups = 4;
struct Pipe {
  cudaStream_t copy_in = nullptr, copy_out = nullptr;
  cudaEvent_t fork = nullptr, join = nullptr, join_out = nullptr, in_ready[kGroups] = {}, out_ready[kGroups] = {};
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
    bool ok = cudaStreamCreateWithFlags(&p.copy_in, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&p.copy_out, cudaStreamNonBlocking) == cudaSuccess &&
              cudaEventCreateWithFlags(&p.fork, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&p.join, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&p.join_out, cudaEventDisableTiming) == cudaSuccess;
    for (int g = 0; g < kGroups && ok; ++g)
      ok = cudaEventCreateWithFlags(&p.in_ready[g], cudaEventDisableTiming) == cudaSuccess &&
           cudaEventCreateWithFlags(&p.out_ready[g], cudaEventDisableTiming) == cudaSuccess;
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
  const size_t step_q = (size_t)Lq * H * d * 2, step_n = (size_t)Ln * H * d * 2;
  const int n_groups = (H % kGroups == 0 && H >= 2 * kGroups) ? kGroups : 1;
  const int32_t Hg = H / n_groups;
  const size_t row_b = (size_t)d * 2, tok_b = row_b * H, grp_b = row_b * Hg;
  const int32_t q_end = Lq, kv_vis = (int32_t)(cache_len_after + Ln);
  ws_block_mask mask{1, &q_end, &kv_vis};
  for (int g = 0; g < n_groups; ++g) {
    const char* kc_g = static_cast<const char*>(k_cache) + (size_t)g * Hg * capacity * row_b;
    const char* vc_g = static_cast<const char*>(v_cache) + (size_t)g * Hg * capacity * row_b;
    if (n_slice_rows > 0)
      if (const int rc = wsi::cache_write_validate(kc_g, vc_g, capacity, Hg, d, st + s.k_slice, st + s.v_slice, n_slice_rows, H, g * Hg,
                                                   row_offset, WS_DTYPE_BF16))
        return rc;
    const size_t off = (size_t)g * grp_b;
    if (const int rc = wsi::attn_validate(st + s.out + off, nullptr, st + s.q + off, kc_g, vc_g, capacity, cache_len_after,
                                          Ln ? st + s.k_new + off : nullptr, Ln ? st + s.v_new + off : nullptr, Ln, Hg, d, Lq, &mask,
                                          softmax_scale, st + s.attn_ws, s.attn_ws_bytes, WS_DTYPE_BF16))
      return rc;
  }

  // ---- pipeline over head groups ----
  // The unit is PCIe-bound (cfg3: 50.8 MB in, 9.9 MB out against 0.27 ms of kernels).  Heads are independent, so the
  // heads are cut into groups: group g's inputs travel as 2-D copies (one head group of every token row) on an
  // internal copy stream, its cache write and attention run on `stream` as soon as they have landed (the fused
  // token-major call reads the group's heads in place), and its output goes home on a second internal stream while
  // the next groups are still arriving.  Everything is joined back into `stream` before the call returns -- also
  // when a later step fails (WS_ERR_CUDA), so a failed call never leaves a stream capture unjoined.
  Pipe* pipe = get_pipe();
  if (!pipe) return wsi::cuda_fail(cudaErrorUnknown);
  // One set of events per device: calls on the same device are serialised on the host for the length of the enqueue.
  std::lock_guard<std::mutex> enqueue_lock(pipe->enqueue_mu);
  // measured on cfg3 (B200, PCIe Gen5): 1 group 1.41 ms per unit, 2 -> 1.28, 4 -> 1.21, 5 -> 1.20, 8 -> 1.27
  cudaError_t e = cudaEventRecord(pipe->fork, stream);
  if (e != cudaSuccess) return wsi::cuda_fail(e);  // nothing has been forked yet
  int rc = WS_OK;
  e = cudaStreamWaitEvent(pipe->copy_in, pipe->fork, 0);
  const bool in_forked = e == cudaSuccess;
  if (e == cudaSuccess) e = cudaStreamWaitEvent(pipe->copy_out, pipe->fork, 0);
  const bool out_forked = in_forked && e == cudaSuccess;
  auto h2d_group = [&](size_t dst_off, const void* src, size_t rows, int g) {
    if (e != cudaSuccess || rows == 0) return;
    e = cudaMemcpy2DAsync(st + dst_off + g * grp_b, tok_b, static_cast<const char*>(src) + g * grp_b, tok_b, grp_b, rows,
                          cudaMemcpyHostToDevice, pipe->copy_in);
  };
  for (int g = 0; g < n_groups && e == cudaSuccess; ++g) {
    h2d_group(s.k_slice, k_slice_host, (size_t)n_slice_rows, g);
    h2d_group(s.v_slice, v_slice_host, (size_t)n_slice_rows, g);
    h2d_group(s.q, q_host, (size_t)n_steps * Lq, g);
    h2d_group(s.k_new, k_new_host, (size_t)n_steps * Ln, g);
    h2d_group(s.v_new, v_new_host, (size_t)n_steps * Ln, g);
    if (e == cudaSuccess) e = cudaEventRecord(pipe->in_ready[g], pipe->copy_in);
  }
  for (int g = 0; g < n_groups && e == cudaSuccess && rc == WS_OK; ++g) {
    e = cudaStreamWaitEvent(stream, pipe->in_ready[g], 0);
    if (e != cudaSuccess) break;
    char* kc_g = static_cast<char*>(k_cache) + (size_t)g * Hg * capacity * row_b;
    char* vc_g = static_cast<char*>(v_cache) + (size_t)g * Hg * capacity * row_b;
    if (n_slice_rows > 0)
      rc = ws_kv_cache_write(kc_g, vc_g, capacity, Hg, d, st + s.k_slice, st + s.v_slice, n_slice_rows, H, g * Hg, row_offset,
                             WS_DTYPE_BF16, stream);
    for (int32_t step = 0; step < n_steps && rc == WS_OK; ++step)
      rc = ws_block_causal_attn_seq_layout(st + s.out + step * step_q, nullptr, st + s.q + step * step_q, kc_g, vc_g, capacity,
                                           cache_len_after, Ln ? st + s.k_new + step * step_n : nullptr,
                                           Ln ? st + s.v_new + step * step_n : nullptr, Ln, H, g * Hg, Hg, d, Lq, &mask,
                                           softmax_scale, st + s.attn_ws, s.attn_ws_bytes, WS_DTYPE_BF16, stream);
    if (rc != WS_OK) break;
    e = cudaEventRecord(pipe->out_ready[g], stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(pipe->copy_out, pipe->out_ready[g], 0);
    if (e == cudaSuccess)
      e = cudaMemcpy2DAsync(static_cast<char*>(out_host) + g * grp_b, tok_b, st + s.out + g * grp_b, tok_b, grp_b, (size_t)n_steps * Lq,
                            cudaMemcpyDeviceToHost, pipe->copy_out);
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
