// ws_fp8.cu -- a1 for the FP8 K/V cache (include/ws.h ws_kv_cache_write_fp8; PAPER.md:79
// "local shards of the full-history cache").
//
//   cache8[h, row_offset + r, :], exp[h, row_offset + r] = quantise(src[r, head_begin + h, :])
//
// quantise (R17/R18): amax = max |x| over the row's d elements; e = the smallest integer with
// 448 * 2^e >= amax, clamped to [-100, 7]; code = RN-even(x / 2^e) to OCP FP8 E4M3, saturated to +-448.
// Roofline: HBM; algorithmic bytes per (row, head) = 2 d read + d + 1 written.  One group of d / 8 lanes per
// (row, head), four groups per thread with their loads issued together: a 16-byte load per lane, the row maximum by shuffles on the BF16 bit patterns (no float math: |x| is
// monotone in its bits), the hardware FP32 -> E4M3 conversion, one 8-byte store per lane (a full 128-byte line per
// row at d = 128).
#include <cuda_bf16.h>

#include "ws_internal.h"

namespace {

constexpr int kThreads = 256;

struct Fp8WriteArgs {
  const uint4* src[2];   // K, V slices, already offset to head_begin
  uint2* cache[2];       // already offset to row_offset
  int8_t* exps[2];       // already offset to row_offset
  int64_t capacity;
  int32_t H, H_src, n_rows;
};

__device__ __forceinline__ uint32_t cvt_e4m3x2(float hi, float lo) {  // {lo -> bits [0,8), hi -> bits [8,16)}
  uint16_t r;
  asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(hi), "f"(lo));
  return r;
}

constexpr int kUnroll = 4;  // (row, head) groups per lane group: four independent 16-byte loads in flight per thread

template <int D>
__global__ void __launch_bounds__(kThreads) kv_write_fp8_kernel(const __grid_constant__ Fp8WriteArgs a) {
  constexpr int kLanes = D / 8;  // lanes per (row, head) group
  constexpr int kGroups = kThreads / kLanes;
  wsi::pdl_trigger();
  const int which = blockIdx.y;
  const int sub = threadIdx.x % kLanes;
  const int64_t n_groups = (int64_t)a.n_rows * a.H;
  int64_t r[kUnroll];
  int h[kUnroll];
  bool active[kUnroll];
#pragma unroll
  for (int u = 0; u < kUnroll; ++u) {
    const int64_t g = ((int64_t)blockIdx.x * kUnroll + u) * kGroups + threadIdx.x / kLanes;  // group = r * H + h: source order
    active[u] = g < n_groups;
    r[u] = active[u] ? g / a.H : 0;
    h[u] = active[u] ? (int)(g - r[u] * a.H) : 0;
  }
  wsi::pdl_wait();  // first global access below
  uint4 v[kUnroll];
#pragma unroll
  for (int u = 0; u < kUnroll; ++u) {
    v[u] = make_uint4(0u, 0u, 0u, 0u);
    if (active[u]) v[u] = a.src[which][(r[u] * a.H_src + h[u]) * kLanes + sub];
  }
#pragma unroll
  for (int u = 0; u < kUnroll; ++u) {
    const uint32_t w[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
    // row maximum of |x| on the bit patterns
    uint32_t amax = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) amax = max(amax, max(w[i] & 0x7fffu, (w[i] >> 16) & 0x7fffu));
#pragma unroll
    for (int off = kLanes / 2; off > 0; off >>= 1) amax = max(amax, __shfl_xor_sync(0xffffffffu, amax, off));
    // amax = 1.m * 2^E (BF16: 8 exponent bits, 7 mantissa bits); 448 = 1.75 * 2^8, so 448 * 2^e >= amax <=> e >= E - 8 (+ 1 if 1.m > 1.75)
    int e = -100;
    if ((amax >> 7) != 0) {  // a subnormal or zero maximum falls below the lower clamp
      e = (int)(amax >> 7) - 127 - 8 + ((amax & 0x7fu) > 0x60u ? 1 : 0);
      e = e < -100 ? -100 : (e > 7 ? 7 : e);
    }
    const float inv = __uint_as_float((uint32_t)(127 - e) << 23);  // 2^-e, exact
    uint32_t out[2];
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const float x0 = __uint_as_float(w[2 * i] << 16) * inv, x1 = __uint_as_float(w[2 * i] & 0xffff0000u) * inv;
      const float x2 = __uint_as_float(w[2 * i + 1] << 16) * inv, x3 = __uint_as_float(w[2 * i + 1] & 0xffff0000u) * inv;
      out[i] = cvt_e4m3x2(x1, x0) | (cvt_e4m3x2(x3, x2) << 16);
    }
    if (active[u]) {
      a.cache[which][((int64_t)h[u] * a.capacity + r[u]) * kLanes + sub] = make_uint2(out[0], out[1]);
      if (sub == 0) a.exps[which][(int64_t)h[u] * a.capacity + r[u]] = (int8_t)e;
    }
  }
}

}  // namespace

extern "C" __attribute__((visibility("default"))) int ws_kv_cache_write_fp8(void* k_cache8, void* v_cache8, int8_t* k_exp, int8_t* v_exp, int64_t capacity, int32_t H,
                                     int32_t d, const void* k_src, const void* v_src, int32_t n_rows, int32_t H_src,
                                     int32_t head_begin, int64_t row_offset, void* stream) {
  if (d != 64 && d != 128) return WS_ERR_UNSUPPORTED;
  if (!k_cache8 || !v_cache8 || !k_exp || !v_exp || capacity <= 0 || H <= 0 || n_rows < 0 || H_src <= 0 || head_begin < 0 ||
      head_begin + (int64_t)H > H_src)
    return WS_ERR_INVALID_ARG;
  if (n_rows > 0 && (!k_src || !v_src)) return WS_ERR_INVALID_ARG;
  if (row_offset < 0 || row_offset + n_rows > capacity) return WS_ERR_OUT_OF_RANGE;
  if (!wsi::aligned16(k_cache8) || !wsi::aligned16(v_cache8) || !wsi::aligned16(k_src) || !wsi::aligned16(v_src) ||
      !wsi::aligned16(k_exp) || !wsi::aligned16(v_exp) || capacity % 16 != 0)
    return WS_ERR_ALIGNMENT;
  if (n_rows == 0) return WS_OK;
  const size_t cache_bytes = (size_t)H * capacity * d, exp_bytes = (size_t)H * capacity, src_bytes = (size_t)n_rows * H_src * d * 2;
  const void* outs[4] = {k_cache8, v_cache8, k_exp, v_exp};
  const size_t out_bytes[4] = {cache_bytes, cache_bytes, exp_bytes, exp_bytes};
  for (int i = 0; i < 4; ++i) {
    if (wsi::ranges_overlap(outs[i], out_bytes[i], k_src, src_bytes) || wsi::ranges_overlap(outs[i], out_bytes[i], v_src, src_bytes))
      return WS_ERR_OVERLAP;
    for (int j = i + 1; j < 4; ++j)
      if (wsi::ranges_overlap(outs[i], out_bytes[i], outs[j], out_bytes[j])) return WS_ERR_OVERLAP;
  }
  const int64_t groups = (int64_t)n_rows * H, per_cta = (int64_t)kUnroll * (kThreads / (d / 8));
  const int64_t blocks = (groups + per_cta - 1) / per_cta;
  if (blocks > 0x7fffffffLL) return WS_ERR_UNSUPPORTED;
  Fp8WriteArgs a;
  a.src[0] = reinterpret_cast<const uint4*>(static_cast<const char*>(k_src) + (int64_t)head_begin * d * 2);
  a.src[1] = reinterpret_cast<const uint4*>(static_cast<const char*>(v_src) + (int64_t)head_begin * d * 2);
  a.cache[0] = reinterpret_cast<uint2*>(static_cast<char*>(k_cache8) + row_offset * d);
  a.cache[1] = reinterpret_cast<uint2*>(static_cast<char*>(v_cache8) + row_offset * d);
  a.exps[0] = k_exp + row_offset;
  a.exps[1] = v_exp + row_offset;
  a.capacity = capacity;
  a.H = H; a.H_src = H_src; a.n_rows = n_rows;
  const dim3 grid((unsigned)blocks, 2);
  const cudaError_t e = d == 128 ? wsi::launch_pdl(kv_write_fp8_kernel<128>, grid, dim3(kThreads), 0, (cudaStream_t)stream, a)
                                 : wsi::launch_pdl(kv_write_fp8_kernel<64>, grid, dim3(kThreads), 0, (cudaStream_t)stream, a);
  if (e != cudaSuccess) return wsi::cuda_fail(e);
  return wsi::after_launch(1);
}
