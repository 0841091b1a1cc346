// ws_copy.cu -- the three HBM-bound byte movers of the hot path, one kernel.
//
//   ws_kv_cache_write  slice [n, H_src, d]  -> cache [H, capacity, d]
//   ws_seq_to_head       [n_tok, H, d]        -> [G, n_tok, H/P, d]
//   ws_head_to_seq       inverse
//
// All three are "copy A x B chunks of dv 16-byte vectors, with independent (a, b) strides on the
// two sides".  Roofline: HBM; algorithmic bytes = payload read once + written once.  The kernel
// keeps 2 independent 16-byte loads in flight per thread (8 KB/CTA, many CTAs per SM), reads with
// ld.global.nc.L1::no_allocate (streamed once) and writes with plain st.global so the freshly
// written cache rows / relaid tensors stay in the 126 MB L2 for the attention kernel that follows.
#include "ws_internal.h"

namespace {

// 256 threads x 2 vectors: measured on B200 over threads in {64..512} x vectors in {1..16} (CUDA-graph timed, rotating
// buffers): small CTAs start streaming sooner on the 5-40 MB moves of the hot path (4.7 MB relayout 3.4 -> 2.3 us,
// 18.8 MB 4.7 -> 4.4 us) and lose nothing on the bandwidth-saturating ones (301 MB: 47.1 -> 46.8 us).
constexpr int kThreads = 256;
constexpr int kUnroll = 2;  // 16-byte vectors per thread

constexpr int kMaxTensors = 4;   // tensors of one *_multi call (ws.h)
constexpr int kMaxEntries = 16;  // (source, destination) pairs moved by one launch (blockIdx.z): tensors x peers
struct CopyPtrs {
  const uint4* src[kMaxEntries];
  uint4* dst[kMaxEntries];
};

struct CopyPlan {
  uint32_t dv;     // 16-byte vectors per contiguous chunk
  uint32_t per_a;  // B * dv: vectors per outer index a
  int64_t src_a, src_b, dst_a, dst_b;  // strides in 16-byte vectors
};

__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

// grid = (ceil(per_a / (kThreads*kUnroll)), A, n_tensors)
__global__ void __launch_bounds__(kThreads) strided_copy16_kernel(const __grid_constant__ CopyPtrs ptrs, const __grid_constant__ CopyPlan p) {
  wsi::pdl_trigger();  // the next kernel may be scheduled now; it blocks in its own pdl_wait() until this grid is done
  const uint4* __restrict__ src = ptrs.src[blockIdx.z];
  uint4* __restrict__ dst = ptrs.dst[blockIdx.z];
  const int64_t a = blockIdx.y;
  src += a * p.src_a;
  dst += a * p.dst_a;
  const uint32_t base = blockIdx.x * (kThreads * kUnroll) + threadIdx.x;
  uint4 v[kUnroll];
  int64_t soff[kUnroll], doff[kUnroll];
#pragma unroll
  for (int u = 0; u < kUnroll; ++u) {
    const uint32_t idx = base + u * kThreads;
    doff[u] = -1;
    if (idx < p.per_a) {
      const uint32_t b = idx / p.dv;
      const uint32_t c = idx - b * p.dv;
      soff[u] = (int64_t)b * p.src_b + c;
      doff[u] = (int64_t)b * p.dst_b + c;
    }
  }
  wsi::pdl_wait();  // first global access below: the previous kernel on the stream has completed
#pragma unroll
  for (int u = 0; u < kUnroll; ++u)
    if (doff[u] >= 0) v[u] = ld_stream(src + soff[u]);
#pragma unroll
  for (int u = 0; u < kUnroll; ++u)
    if (doff[u] >= 0) dst[doff[u]] = v[u];
}

// Launches the plan for n_tensors (source, destination) pairs of the same shape, splitting B so that per_a stays below 2^30 vectors.
int launch_copy(const void* const* srcs, void* const* dsts, int n_tensors, int64_t A, int64_t B, int64_t dv, int64_t src_a,
                int64_t src_b, int64_t dst_a, int64_t dst_b, cudaStream_t stream) {
  if (A == 0 || B == 0 || dv == 0 || n_tensors == 0) return WS_OK;
  if (A > 65535 || dv > (1 << 20) || n_tensors > kMaxEntries) return WS_ERR_UNSUPPORTED;
  const int64_t max_b = ((int64_t)1 << 30) / dv;
  int launches = 0;
  for (int64_t b0 = 0; b0 < B; b0 += max_b) {
    const int64_t nb = (B - b0 < max_b) ? (B - b0) : max_b;
    CopyPlan p;
    p.dv = (uint32_t)dv;
    p.per_a = (uint32_t)(nb * dv);
    p.src_a = src_a; p.src_b = src_b; p.dst_a = dst_a; p.dst_b = dst_b;
    CopyPtrs ptrs = {};
    for (int i = 0; i < n_tensors; ++i) {
      ptrs.src[i] = reinterpret_cast<const uint4*>(srcs[i]) + b0 * src_b;
      ptrs.dst[i] = reinterpret_cast<uint4*>(dsts[i]) + b0 * dst_b;
    }
    dim3 grid((unsigned)((p.per_a + kThreads * kUnroll - 1) / (kThreads * kUnroll)), (unsigned)A, (unsigned)n_tensors);
    const cudaError_t e = wsi::launch_pdl(strided_copy16_kernel, grid, dim3(kThreads), 0, stream, ptrs, p);
    if (e != cudaSuccess) return wsi::cuda_fail(e);
    ++launches;
  }
  return wsi::after_launch(launches);
}

int relayout(void* const* dsts, const void* const* srcs, int n_tensors, int64_t n_tok, int32_t H, int32_t d, int32_t P, int32_t g0,
             int32_t G, ws_dtype dt, void* stream, bool to_head) {
  const int es = wsi::elem_bytes(dt);
  if (es == 0) return WS_ERR_UNSUPPORTED;
  if (!dsts || !srcs || n_tensors < 0 || n_tok < 0 || H <= 0 || d <= 0 || P <= 0 || H % P != 0 || g0 < 0 || G < 0 || g0 + G > P)
    return WS_ERR_INVALID_ARG;
  if (n_tensors > kMaxTensors) return WS_ERR_UNSUPPORTED;
  const int32_t Hp = H / P;
  const int64_t chunk_bytes = (int64_t)Hp * d * es;  // contiguous bytes per (g, t)
  if (((int64_t)d * es) % 16 != 0) return WS_ERR_ALIGNMENT;
  const size_t tok_bytes = (size_t)n_tok * H * d * es;          // token-major tensor
  const size_t head_bytes = (size_t)G * n_tok * chunk_bytes;    // head-major tensor
  const size_t dst_bytes = to_head ? head_bytes : tok_bytes, src_bytes = to_head ? tok_bytes : head_bytes;
  for (int i = 0; i < n_tensors; ++i) {
    if (!dsts[i] || !srcs[i]) return WS_ERR_INVALID_ARG;
    if (!wsi::aligned16(dsts[i]) || !wsi::aligned16(srcs[i])) return WS_ERR_ALIGNMENT;
  }
  for (int i = 0; i < n_tensors; ++i) {  // no destination may intersect any source or any other destination
    for (int j = 0; j < n_tensors; ++j) {
      if (wsi::ranges_overlap(dsts[i], dst_bytes, srcs[j], src_bytes)) return WS_ERR_OVERLAP;
      if (j != i && wsi::ranges_overlap(dsts[i], dst_bytes, dsts[j], dst_bytes)) return WS_ERR_OVERLAP;
    }
  }
  const int64_t dv = chunk_bytes / 16;
  const int64_t tok_a = (int64_t)Hp * d * es / 16;   // token-major: group g -> + g * Hp heads
  const int64_t tok_b = (int64_t)H * d * es / 16;    // token t
  const int64_t head_a = n_tok * dv;                 // head-major: group g
  const int64_t head_b = dv;                         // token t
  const void* s2[kMaxTensors];
  void* d2[kMaxTensors];
  for (int i = 0; i < n_tensors; ++i) {  // the token-major side starts at the first selected head group
    s2[i] = to_head ? static_cast<const void*>(reinterpret_cast<const char*>(srcs[i]) + (int64_t)g0 * chunk_bytes) : srcs[i];
    d2[i] = to_head ? dsts[i] : static_cast<void*>(reinterpret_cast<char*>(dsts[i]) + (int64_t)g0 * chunk_bytes);
  }
  if (to_head) return launch_copy(s2, d2, n_tensors, G, n_tok, dv, tok_a, tok_b, head_a, head_b, (cudaStream_t)stream);
  return launch_copy(s2, d2, n_tensors, G, n_tok, dv, head_a, head_b, tok_a, tok_b, (cudaStream_t)stream);
}

}  // namespace

// Every argument check of ws_kv_cache_write (host only; see ws_internal.h).
int wsi::cache_write_validate(const void* k_cache, const void* v_cache, int64_t capacity, int32_t H, int32_t d, const void* k_src,
                              const void* v_src, int32_t n_rows, int32_t H_src, int32_t head_begin, int64_t row_offset, ws_dtype dt) {
  const int es = wsi::elem_bytes(dt);
  if (es == 0) return WS_ERR_UNSUPPORTED;
  if (!k_cache || !v_cache || capacity <= 0 || H <= 0 || d <= 0 || n_rows < 0 || H_src <= 0 || head_begin < 0 ||
      head_begin + (int64_t)H > H_src)
    return WS_ERR_INVALID_ARG;
  if (n_rows > 0 && (!k_src || !v_src)) return WS_ERR_INVALID_ARG;
  if (row_offset < 0 || row_offset + n_rows > capacity) return WS_ERR_OUT_OF_RANGE;
  const int64_t row_bytes = (int64_t)d * es;
  if (row_bytes % 16 != 0 || !wsi::aligned16(k_cache) || !wsi::aligned16(v_cache) || !wsi::aligned16(k_src) ||
      !wsi::aligned16(v_src))
    return WS_ERR_ALIGNMENT;
  if (H > 65535 || row_bytes / 16 > (1 << 20)) return WS_ERR_UNSUPPORTED;  // launch_copy's limits
  if (n_rows == 0) return WS_OK;
  const size_t cache_bytes = (size_t)H * capacity * row_bytes, src_bytes = (size_t)n_rows * H_src * row_bytes;
  const void* caches[2] = {k_cache, v_cache};
  const void* srcs[2] = {k_src, v_src};
  for (int i = 0; i < 2; ++i)
    for (int j = 0; j < 2; ++j)
      if (wsi::ranges_overlap(caches[i], cache_bytes, srcs[j], src_bytes)) return WS_ERR_OVERLAP;
  if (wsi::ranges_overlap(k_cache, cache_bytes, v_cache, cache_bytes)) return WS_ERR_OVERLAP;
  return WS_OK;
}

extern "C" __attribute__((visibility("default"))) int ws_kv_cache_write(void* k_cache, void* v_cache, int64_t capacity, int32_t H, int32_t d, const void* k_src,
                                 const void* v_src, int32_t n_rows, int32_t H_src, int32_t head_begin, int64_t row_offset,
                                 ws_dtype dt, void* stream) {
  if (const int rc = wsi::cache_write_validate(k_cache, v_cache, capacity, H, d, k_src, v_src, n_rows, H_src, head_begin, row_offset, dt))
    return rc;
  if (n_rows == 0) return WS_OK;
  const int64_t row_bytes = (int64_t)d * wsi::elem_bytes(dt);
  const int64_t dv = row_bytes / 16;
  // a = head h, b = row r:  src (r * H_src + head_begin + h) * dv ; dst (h * capacity + row_offset + r) * dv
  const char* ks = reinterpret_cast<const char*>(k_src) + (int64_t)head_begin * row_bytes;
  const char* vs = reinterpret_cast<const char*>(v_src) + (int64_t)head_begin * row_bytes;
  char* kd = reinterpret_cast<char*>(k_cache) + row_offset * row_bytes;
  char* vd = reinterpret_cast<char*>(v_cache) + row_offset * row_bytes;
  const void* srcs2[2] = {ks, vs};
  void* dsts2[2] = {kd, vd};
  return launch_copy(srcs2, dsts2, 2, H, n_rows, dv, dv, (int64_t)H_src * dv, capacity * dv, dv, (cudaStream_t)stream);
}

// Ring (sliding-window) cache write, SURVEY.md 8(f).4 / DESIGN.md R19: session row write_pos + r goes to physical row
// (write_pos + r) mod capacity.  At most two physical runs: one launch each (the second only when the slice wraps).
extern "C" __attribute__((visibility("default"))) int ws_kv_cache_write_ring(void* k_cache, void* v_cache, int64_t capacity, int32_t H, int32_t d, const void* k_src,
                                      const void* v_src, int32_t n_rows, int32_t H_src, int32_t head_begin, int64_t write_pos,
                                      ws_dtype dt, void* stream) {
  if (write_pos < 0 || capacity <= 0) return capacity <= 0 ? WS_ERR_INVALID_ARG : WS_ERR_OUT_OF_RANGE;
  if (n_rows > capacity) return WS_ERR_OUT_OF_RANGE;  // a call never overwrites a row it has written itself
  const int64_t phys = write_pos % capacity;
  const int64_t n_a = n_rows < capacity - phys ? n_rows : capacity - phys, n_b = n_rows - n_a;
  // both runs are checked before the first launch (the second run starts at physical row 0 with the slice's rows n_a ..)
  if (const int rc = wsi::cache_write_validate(k_cache, v_cache, capacity, H, d, k_src, v_src, n_rows, H_src, head_begin, n_b > 0 ? 0 : phys, dt))
    return rc;
  if (n_rows == 0) return WS_OK;
  const int64_t row_bytes = (int64_t)d * wsi::elem_bytes(dt), dv = row_bytes / 16;
  int rc = WS_OK;
  for (int run = 0; run < 2 && rc == WS_OK; ++run) {
    const int64_t n = run ? n_b : n_a, dst_row = run ? 0 : phys, src_row = run ? n_a : 0;
    if (n == 0) continue;
    const void* srcs2[2] = {reinterpret_cast<const char*>(k_src) + (src_row * H_src + head_begin) * row_bytes,
                            reinterpret_cast<const char*>(v_src) + (src_row * H_src + head_begin) * row_bytes};
    void* dsts2[2] = {reinterpret_cast<char*>(k_cache) + dst_row * row_bytes, reinterpret_cast<char*>(v_cache) + dst_row * row_bytes};
    rc = launch_copy(srcs2, dsts2, 2, H, n, dv, dv, (int64_t)H_src * dv, capacity * dv, dv, (cudaStream_t)stream);
  }
  return rc;
}

// ---------------------------------------------------------------------------------------------------------------------
// Ulysses exchange over peer memory.  Push model: the sender's copy kernel stores
// straight into the receivers' buffers through peer-mapped pointers (NVLink / NVSwitch P2P stores; on one GPU the "peers"
// are local buffers), in the layout the attention kernel reads -- the pack (a2) and the transport are one kernel and
// nothing is staged.  blockIdx.z walks the (tensor, peer) pairs.
// ---------------------------------------------------------------------------------------------------------------------
extern "C" __attribute__((visibility("default"))) int ws_ulysses_push_seq_to_head(void* const* peer_dsts, const void* const* srcs, int32_t n_tensors, int64_t Ls,
                                           int64_t La, int32_t H, int32_t d, int32_t P, int32_t rank, ws_dtype dt, void* stream) {
  const int es = wsi::elem_bytes(dt);
  if (es == 0) return WS_ERR_UNSUPPORTED;
  if (!peer_dsts || !srcs || n_tensors < 0 || Ls < 0 || La < 0 || H <= 0 || d <= 0 || P <= 0 || H % P != 0 || rank < 0 || rank >= P)
    return WS_ERR_INVALID_ARG;
  if (n_tensors > kMaxTensors || P > WS_MAX_PEERS) return WS_ERR_UNSUPPORTED;
  if (((int64_t)d * es) % 16 != 0) return WS_ERR_ALIGNMENT;
  const int32_t Hp = H / P;
  const int64_t chunk_bytes = (int64_t)Hp * d * es, dv = chunk_bytes / 16, tok_b = (int64_t)H * d * es / 16;
  const size_t src_bytes = (size_t)(Ls + La) * H * d * es, dst_bytes = (size_t)(P * Ls + La) * chunk_bytes;
  for (int i = 0; i < n_tensors; ++i) {
    if (!srcs[i]) return WS_ERR_INVALID_ARG;
    if (!wsi::aligned16(srcs[i])) return WS_ERR_ALIGNMENT;
    for (int g = 0; g < P; ++g) {
      if (!peer_dsts[i * P + g]) return WS_ERR_INVALID_ARG;
      if (!wsi::aligned16(peer_dsts[i * P + g])) return WS_ERR_ALIGNMENT;
    }
  }
  // unified virtual addressing: a peer-mapped range and a local range intersect only if they are the same memory
  for (int i = 0; i < n_tensors * P; ++i) {
    for (int j = 0; j < n_tensors; ++j)
      if (wsi::ranges_overlap(peer_dsts[i], dst_bytes, srcs[j], src_bytes)) return WS_ERR_OVERLAP;
    for (int j = 0; j < i; ++j)
      if (wsi::ranges_overlap(peer_dsts[i], dst_bytes, peer_dsts[j], dst_bytes)) return WS_ERR_OVERLAP;
  }
  // sharded (video) rows: Y_g[rank * Ls + t, c, :] = X[t, g * Hp + c, :] on every peer g
  const void* s2[kMaxEntries];
  void* d2[kMaxEntries];
  int n = 0, rc = WS_OK;
  for (int i = 0; i < n_tensors && rc == WS_OK; ++i)
    for (int g = 0; g < P && rc == WS_OK; ++g) {
      s2[n] = reinterpret_cast<const char*>(srcs[i]) + (int64_t)g * chunk_bytes;
      d2[n] = reinterpret_cast<char*>(peer_dsts[i * P + g]) + (int64_t)rank * Ls * chunk_bytes;
      if (++n == kMaxEntries || (i == n_tensors - 1 && g == P - 1)) {
        rc = launch_copy(s2, d2, n, 1, Ls, dv, 0, tok_b, 0, dv, (cudaStream_t)stream);
        n = 0;
      }
    }
  // unsharded (audio) rows are replicated on every rank: the rank's own heads are a local relayout
  for (int i = 0; i < n_tensors; ++i) {
    s2[i] = reinterpret_cast<const char*>(srcs[i]) + (Ls * H + (int64_t)rank * Hp) * d * es;
    d2[i] = reinterpret_cast<char*>(peer_dsts[i * P + rank]) + (int64_t)P * Ls * chunk_bytes;
  }
  if (rc == WS_OK) rc = launch_copy(s2, d2, n_tensors, 1, La, dv, 0, tok_b, 0, dv, (cudaStream_t)stream);
  return rc;
}

// The thinker's K/V slice [n_rows, P * Hp, d] written into every performer rank's cache [Hp, capacity, d] by ONE kernel
// (broadcast fused with a1): the slice is read once and each rank's head range is stored through that rank's peer pointer.
extern "C" __attribute__((visibility("default"))) int ws_kv_slice_broadcast_write(void* const* peer_k_caches, void* const* peer_v_caches, int32_t P, int64_t capacity,
                                           int32_t Hp, int32_t d, const void* k_src, const void* v_src, int32_t n_rows,
                                           int64_t row_offset, ws_dtype dt, void* stream) {
  if (!peer_k_caches || !peer_v_caches || P <= 0 || Hp <= 0) return WS_ERR_INVALID_ARG;
  if (P > WS_MAX_PEERS) return WS_ERR_UNSUPPORTED;
  if ((int64_t)P * Hp > 0x7fffffff) return WS_ERR_INVALID_ARG;
  for (int g = 0; g < P; ++g)
    if (const int rc = wsi::cache_write_validate(peer_k_caches[g], peer_v_caches[g], capacity, Hp, d, k_src, v_src, n_rows, P * Hp, g * Hp,
                                                 row_offset, dt))
      return rc;
  const int64_t row_bytes = (int64_t)d * wsi::elem_bytes(dt), dv = row_bytes / 16;
  const size_t cache_bytes = (size_t)Hp * capacity * row_bytes;
  for (int g = 0; g < P; ++g)  // two ranks' caches must not be the same memory
    for (int j = 0; j < g; ++j)
      if (wsi::ranges_overlap(peer_k_caches[g], cache_bytes, peer_k_caches[j], cache_bytes) || wsi::ranges_overlap(peer_v_caches[g], cache_bytes, peer_v_caches[j], cache_bytes) ||
          wsi::ranges_overlap(peer_k_caches[g], cache_bytes, peer_v_caches[j], cache_bytes) || wsi::ranges_overlap(peer_v_caches[g], cache_bytes, peer_k_caches[j], cache_bytes))
        return WS_ERR_OVERLAP;
  if (n_rows == 0) return WS_OK;
  const void* s2[kMaxEntries];
  void* d2[kMaxEntries];
  for (int g = 0; g < P; ++g) {
    s2[2 * g] = reinterpret_cast<const char*>(k_src) + (int64_t)g * Hp * row_bytes;
    s2[2 * g + 1] = reinterpret_cast<const char*>(v_src) + (int64_t)g * Hp * row_bytes;
    d2[2 * g] = reinterpret_cast<char*>(peer_k_caches[g]) + row_offset * row_bytes;
    d2[2 * g + 1] = reinterpret_cast<char*>(peer_v_caches[g]) + row_offset * row_bytes;
  }
  static_assert(2 * WS_MAX_PEERS <= kMaxEntries, "one launch holds K and V of every peer");
  return launch_copy(s2, d2, 2 * P, Hp, n_rows, dv, dv, (int64_t)P * Hp * dv, capacity * dv, dv, (cudaStream_t)stream);
}

// The window after rows_written rows of the session (host only): cache_len = min(rows_written, capacity) valid rows, the
// oldest of which sits in physical row ring_start.
extern "C" __attribute__((visibility("default"))) int ws_ring_state(int64_t rows_written, int64_t capacity, int64_t* ring_start, int64_t* cache_len) {
  if (rows_written < 0 || capacity <= 0 || !ring_start || !cache_len) return WS_ERR_INVALID_ARG;
  *ring_start = rows_written < capacity ? 0 : rows_written % capacity;
  *cache_len = rows_written < capacity ? rows_written : capacity;
  return WS_OK;
}

extern "C" __attribute__((visibility("default"))) int ws_seq_to_head(void* dst, const void* src, int64_t n_tok, int32_t H, int32_t d, int32_t P, int32_t g0, int32_t G,
                              ws_dtype dt, void* stream) {
  return relayout(&dst, &src, 1, n_tok, H, d, P, g0, G, dt, stream, true);
}

extern "C" __attribute__((visibility("default"))) int ws_head_to_seq(void* dst, const void* src, int64_t n_tok, int32_t H, int32_t d, int32_t P, int32_t g0, int32_t G,
                              ws_dtype dt, void* stream) {
  return relayout(&dst, &src, 1, n_tok, H, d, P, g0, G, dt, stream, false);
}

// Several tensors of one shape in ONE launch (Q, K_new and V_new before attention): the launch and DRAM round-trip
// latency that dominates a 10-20 MB relayout is paid once.
extern "C" __attribute__((visibility("default"))) int ws_seq_to_head_multi(void* const* dsts, const void* const* srcs, int32_t n_tensors, int64_t n_tok,
                                    int32_t H, int32_t d, int32_t P, int32_t g0, int32_t G, ws_dtype dt, void* stream) {
  return relayout(dsts, srcs, n_tensors, n_tok, H, d, P, g0, G, dt, stream, true);
}

extern "C" __attribute__((visibility("default"))) int ws_head_to_seq_multi(void* const* dsts, const void* const* srcs, int32_t n_tensors, int64_t n_tok,
                                    int32_t H, int32_t d, int32_t P, int32_t g0, int32_t G, ws_dtype dt, void* stream) {
  return relayout(dsts, srcs, n_tensors, n_tok, H, d, P, g0, G, dt, stream, false);
}
