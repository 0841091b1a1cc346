/*
 * ws.h -- C ABI of the B200-native performer hot path of Wan-Streamer v0.2
 *         (arxiv/paper_2607_04443; citations are PAPER.md line numbers).
 *
 * One Ulysses performer rank's single-GPU share of a 160 ms streaming unit:
 *
 *   ws_kv_cache_write      "each performer rank writes incoming K/V into a pre-sharded local
 *                           cache"
 *   ws_seq_to_head /       the rank-local halves of the "Ulysses all-to-all/gather collectives
 *   ws_head_to_seq          around attention"
 *   ws_block_causal_attn   the unit's latent query tokens attend, "coordinated by block-causal
 *                           attention", to the cached K/V conditioning plus the unit's own K/V
 *                                                                   PAPER.md:25, :73, :79
 *   ws_block_causal_attn_static_ws    a3 for callers that cannot allocate device memory: the scratch is an array
 *                           inside the library's own device image (at most WS_STATIC_WORKSPACE_BYTES)
 *   ws_block_causal_attn_seq_layout   the two relayouts folded into the attention call (strided TMA)
 *   ws_seq_to_head_multi / ws_head_to_seq_multi   several same-shaped tensors in one launch
 *   ws_kv_cache_write_fp8 / ws_block_causal_attn_fp8kv   the same cache held as FP8 (E4M3 codes and one
 *                           power-of-two scale per (row, head)): half the bytes of the full-history cache
 *   ws_kv_cache_write_ring / ws_block_causal_attn_ring / ws_ring_state   the cache as a sliding window over an
 *                           unbounded session: a ring that keeps the most recent `capacity` rows
 *   ws_ulysses_push_seq_to_head / ws_block_causal_attn_push_out / ws_kv_slice_broadcast_write   the exchanges of a
 *                           multi-GPU Ulysses performer group done as stores into peer memory (NVLink P2P) by the
 *                           pack kernel, the attention epilogue and the cache-write kernel themselves
 *   ws_unit_forward_host   the same path for one unit fed from HOST buffers (end-to-end entry)
 *   ws_attn_schedule       host-only diagnostic: the attention work schedule for a given SM count
 *
 * Conventions (all functions)
 *   - Return value: WS_OK (0) or a negative ws_status.  Every argument is checked, every TMA
 *     descriptor encoded and the work schedule built BEFORE the first launch or copy: on any
 *     argument error (every status except WS_ERR_CUDA) NOTHING is launched, nothing is enqueued
 *     and no output byte is modified.  WS_ERR_CUDA (the cudaError_t is kept in
 *     ws_last_cuda_error()) reports a failure of the CUDA runtime itself; if it strikes in the
 *     middle of a multi-launch call the earlier launches stay enqueued and outputs are undefined.
 *   - Per-device state (SM count, kernel attributes, a5's helper streams) is keyed by the current
 *     device: one process may drive several GPUs (cudaSetDevice before the call).
 *   - Pointers documented "device" are CUDA device pointers OWNED BY THE CALLER and borrowed
 *     until the stream-ordered work completes.  Pointers documented "host" are read during the
 *     call only.  Device pointers must be 16-byte aligned and d * sizeof(element) a multiple of
 *     16 (WS_ERR_ALIGNMENT otherwise).
 *   - No allocation, no synchronisation, no host read of device data: every call is legal
 *     inside CUDA stream capture (this sentence does not cover ws_block_causal_attn_static_ws, which says
 *     when its first call on a device must come).  `stream` is a cudaStream_t passed as void* (NULL = default).
 *     Kernels are launched with programmatic stream serialisation (their set-up overlaps the tail
 *     of the previous kernel; they wait for it before touching global memory).
 *   - Batch is 1 (fold a batch into heads).  Layouts are dense row-major with the last index
 *     fastest: token-major [L, H, d] for Q / K_new / V_new / O / slices, head-major
 *     [H, capacity, d] for the cache (private to the rank; reading R5).
 *   - There is no CPU fallback: without a CUDA device every launching call fails.
 */
#ifndef WS_H_
#define WS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* major*10000 + minor*100 + patch.  0.1.0: rows a1-a5.  0.2.0: ws_attn_schedule gained unit_kv_tiles (NOT call-compatible
 * with 0.1.0), FP8 / ring / Ulysses entry points.  0.3.0: ws_block_causal_attn_static_ws, overlap rules of push_out / fp8kv. */
#define WS_VERSION 300

typedef enum { WS_DTYPE_BF16 = 0, WS_DTYPE_F32 = 1 } ws_dtype;

typedef enum {
  WS_OK = 0,
  WS_ERR_INVALID_ARG = -1,  /* NULL pointer, non-positive size, malformed mask, H % P != 0 ...   */
  WS_ERR_UNSUPPORTED = -2,  /* dtype / head_dim / mask size this build has no kernel for         */
  WS_ERR_ALIGNMENT = -3,    /* a device pointer or row pitch is not 16-byte aligned              */
  WS_ERR_OUT_OF_RANGE = -4, /* row_offset+n_rows > capacity, cache_len > capacity, kv_visible > cache_len+Ln */
  WS_ERR_OVERLAP = -5,      /* source and destination byte ranges intersect                      */
  WS_ERR_WORKSPACE = -6,    /* workspace NULL or smaller than ws_block_causal_attn_workspace_bytes */
  WS_ERR_CUDA = -7          /* CUDA runtime/driver error; see ws_last_cuda_error()               */
} ws_status;

/* Limits of this build. */
#define WS_MAX_MASK_BLOCKS 128 /* n_blocks of a ws_block_mask */
#define WS_MAX_PEERS 8         /* ranks of a Ulysses performer group (ws_ulysses_*, ws_block_causal_attn_push_out) */
#define WS_STATIC_WORKSPACE_BYTES (64u << 20) /* scratch built into the library for ws_block_causal_attn_static_ws */

/* ------------------------------------------------------------------------------------------------
 * a1. KV cache write
 *
 *   cache[h, row_offset + r, :] = src[r, head_begin + h, :]   0 <= h < H, 0 <= r < n_rows
 *   for K and for V; every other cache byte is untouched.
 *
 *   k_cache, v_cache : device, [H, capacity, d]   (written)
 *   k_src, v_src     : device, [n_rows, H_src, d] (read) -- the thinker's broadcast slice with all
 *                      H_src heads; this rank keeps heads [head_begin, head_begin + H).
 *   n_rows == 0 is a no-op (WS_OK).  Errors: OUT_OF_RANGE if row_offset < 0 or
 *   row_offset + n_rows > capacity; INVALID_ARG if head_begin < 0 or head_begin + H > H_src;
 *   OVERLAP if a source range intersects a cache range.
 * ---------------------------------------------------------------------------------------------- */
int ws_kv_cache_write(void* k_cache, void* v_cache, int64_t capacity, int32_t H, int32_t d,
                      const void* k_src, const void* v_src, int32_t n_rows, int32_t H_src,
                      int32_t head_begin, int64_t row_offset, ws_dtype dt, void* stream);

/* ------------------------------------------------------------------------------------------------
 * a2 / a4. Ulysses-local relayouts
 *
 *   With Hp = H / P heads per rank-group:
 *   ws_seq_to_head:  dst[g, t, c, :] = src[t, (g0 + g) * Hp + c, :]
 *   ws_head_to_seq:  dst[t, (g0 + g) * Hp + c, :] = src[g, t, c, :]   (other heads of dst untouched)
 *   for 0 <= g < G, 0 <= t < n_tok, 0 <= c < Hp.  They are exact inverses on the selected heads.
 *
 *   token-major side : device, [n_tok, H, d]       head-major side : device, [G, n_tok, Hp, d]
 *   G = 1 with g0 = rank is what one rank needs after all-to-all #1 when all sequence shards are
 *   local (config 4); G = P packs every peer's chunk (the send buffer of a real all-to-all).
 *   Errors: INVALID_ARG if P <= 0, H % P != 0, g0 < 0, G < 0 or g0 + G > P; OVERLAP if src and dst
 *   intersect.  n_tok == 0 or G == 0 is a no-op.
 * ---------------------------------------------------------------------------------------------- */
int ws_seq_to_head(void* dst, const void* src, int64_t n_tok, int32_t H, int32_t d, int32_t P,
                   int32_t g0, int32_t G, ws_dtype dt, void* stream);
int ws_head_to_seq(void* dst, const void* src, int64_t n_tok, int32_t H, int32_t d, int32_t P,
                   int32_t g0, int32_t G, ws_dtype dt, void* stream);

/* a2 / a4 on several tensors of one shape in ONE launch (at most 4; e.g. Q, K_new and V_new before
 * attention).  dsts / srcs are HOST arrays of n_tensors device pointers, read during the call only.
 * Semantics, layouts and errors per tensor exactly as ws_seq_to_head / ws_head_to_seq; in addition no
 * destination may intersect any source or any other destination (OVERLAP), and n_tensors > 4 is
 * UNSUPPORTED.  A 10-20 MB relayout is dominated by launch and DRAM round-trip latency:
 * batching pays it once. */
int ws_seq_to_head_multi(void* const* dsts, const void* const* srcs, int32_t n_tensors, int64_t n_tok, int32_t H,
                         int32_t d, int32_t P, int32_t g0, int32_t G, ws_dtype dt, void* stream);
int ws_head_to_seq_multi(void* const* dsts, const void* const* srcs, int32_t n_tensors, int64_t n_tok, int32_t H,
                         int32_t d, int32_t P, int32_t g0, int32_t G, ws_dtype dt, void* stream);

/* ------------------------------------------------------------------------------------------------
 * a3. Block-causal unit attention
 *
 *   Key timeline: j < cache_len is cache row j; cache_len <= j < cache_len + Ln is row
 *   j - cache_len of k_new / v_new.  Query block b covers rows [q_block_end[b-1], q_block_end[b])
 *   (q_block_end[-1] = 0) and sees the keys j < kv_visible[b]:
 *
 *     O[i, h, :] = sum_{j < kv_visible[b(i)]} softmax_j(softmax_scale * q[i,h,:] . k_j[h,:]) v_j[h,:]
 *     lse[h, i]  = natural-log-sum-exp of the visible scaled logits
 *     kv_visible[b] == 0  ->  O row = 0, lse = -inf (no NaN).
 *
 *   A streaming unit is one block (bidirectional inside the unit, causal across units).
 *
 *   out      : device, [Lq, H, d], same dtype as q (written)
 *   lse      : device, float [H, Lq], or NULL
 *   q        : device, [Lq, H, d]
 *   k_cache, v_cache : device, [H, capacity, d]; rows [0, cache_len) are valid and must be finite
 *   k_new, v_new     : device, [Ln, H, d]; NULL iff Ln == 0
 *   mask     : host; q_block_end strictly increasing with last == Lq; kv_visible non-decreasing,
 *              0 <= kv_visible[b] <= cache_len + Ln; n_blocks <= WS_MAX_MASK_BLOCKS
 *   workspace: device, >= ws_block_causal_attn_workspace_bytes(...) bytes, 256-byte aligned;
 *              contents are scratch (split-KV partials; BF16 staging for WS_DTYPE_F32)
 *
 *   Arithmetic: BF16 operands, FP32 accumulation (tcgen05), FP32 softmax, probabilities rounded
 *   to BF16 before P.V.  WS_DTYPE_F32 inputs are rounded to BF16 on the device first and the
 *   output is written as FP32 (config 1; reading R9).  Supported: d in {64, 128}.
 *   Errors: UNSUPPORTED (d, dt, n_blocks), INVALID_ARG (malformed mask, NULLs), OUT_OF_RANGE
 *   (cache_len > capacity, kv_visible > cache_len + Ln), WORKSPACE, ALIGNMENT, CUDA.
 * ---------------------------------------------------------------------------------------------- */
typedef struct ws_block_mask {
  int32_t n_blocks;
  const int32_t* q_block_end; /* host */
  const int32_t* kv_visible;  /* host */
} ws_block_mask;

size_t ws_block_causal_attn_workspace_bytes(int32_t Lq, int32_t H, int32_t d, int64_t kv_total, ws_dtype dt);

int ws_block_causal_attn(void* out, float* lse, const void* q, const void* k_cache, const void* v_cache,
                         int64_t capacity, int64_t cache_len, const void* k_new, const void* v_new, int32_t Ln,
                         int32_t H, int32_t d, int32_t Lq, const ws_block_mask* mask, float softmax_scale,
                         void* workspace, size_t workspace_bytes, ws_dtype dt, void* stream);

/* ------------------------------------------------------------------------------------------------
 * a3 without a caller-supplied workspace: for callers that cannot allocate.
 *
 *   ws_block_causal_attn needs scratch in device memory and leaves it to the caller to provide.  Not every caller
 *   can: a plug-in inside a serving process that handed all of HBM to its framework's pools at start-up (cudaMalloc
 *   fails, the pool is out of reach from C); the per-unit real-time loop, where a cudaMalloc / cudaFree would
 *   synchronise the device and stall the units in flight (one unit per 160 ms); code bound by a
 *   "nothing is allocated after initialisation" rule.  This entry point is ws_block_causal_attn with the scratch
 *   taken from a fixed array of WS_STATIC_WORKSPACE_BYTES (64 MiB) that is part of the library's device image.  It
 *   calls no cudaMalloc, cudaFree or any allocating library routine; the caller passes inputs and outputs only.
 *
 *   Arguments, arithmetic, results and errors are exactly those of ws_block_causal_attn (the same kernels run on the
 *   same schedule), minus `workspace` / `workspace_bytes`.
 *
 *   Limit:  the problem must satisfy  ws_block_causal_attn_workspace_bytes(Lq, H, d, cache_len + Ln, dt)
 *           <= WS_STATIC_WORKSPACE_BYTES, else WS_ERR_WORKSPACE is returned and nothing is launched.  64 MiB covers
 *           every BF16 configuration of BASELINE.json (config 3, 970 x 40 heads x 128: 55.4 MB; the need grows with
 *           ceil(Lq / 256) * H * d and does not depend on the cache length for BF16 inputs).
 *   Cost:   every GPU on which the library's device code is loaded holds the 64 MiB until the process exits, used or not.
 *   First call on a device:  looks up the array's address on that device (cudaGetSymbolAddress, once per device, the
 *           device being current) and remembers it.  Make that first call during set-up, before any stream capture
 *           is begun on that device.
 *   Sharing: every call on a device uses the same array, which still holds whatever the previous call left there.
 *           No part of it has to be zero on entry -- each call writes what it later reads -- so it is never cleared.
 *           Two calls that can overlap on the GPU (different streams, or several host threads launching at once)
 *           race on it and corrupt each other's partial results: keep all calls of a device on one stream, or order
 *           them with events.  (ws_block_causal_attn with separate workspaces has no such restriction.)
 *   Errors: as ws_block_causal_attn; WS_ERR_WORKSPACE means "needs more scratch than the built-in array has";
 *           WS_ERR_CUDA if the address look-up fails.
 * ---------------------------------------------------------------------------------------------- */
int ws_block_causal_attn_static_ws(void* out, float* lse, const void* q, const void* k_cache, const void* v_cache,
                                   int64_t capacity, int64_t cache_len, const void* k_new, const void* v_new, int32_t Ln,
                                   int32_t H, int32_t d, int32_t Lq, const ws_block_mask* mask, float softmax_scale,
                                   ws_dtype dt, void* stream);

/* ------------------------------------------------------------------------------------------------
 * a2 + a3 + a4 fused: attention straight on the token-major layout
 *
 *   The collectives "around attention" exist to hand a rank the full sequence of its own heads.
 *   When that sequence already sits in local memory as token-major [n_tok, H_total, d] tensors
 *   (single GPU; or after a peer has written its tokens in place), the two relayouts are pure
 *   address arithmetic: this call reads the heads [head_begin, head_begin + H) of q_seq,
 *   k_new_seq, v_new_seq through strided TMA descriptors and stores O into the same heads of
 *   out_seq, whose other heads are not touched.  It equals
 *       ws_seq_to_head(q, k_new, v_new) -> ws_block_causal_attn -> ws_head_to_seq(out)
 *   with P = H_total / H, g0 = head_begin / H, G = 1, bit for bit, without the 4 x n_tok x H x d
 *   element round trip through HBM.
 *
 *   out_seq            : device, [Lq, H_total, d]
 *   q_seq              : device, [Lq, H_total, d]
 *   k_new_seq, v_new_seq : device, [Ln, H_total, d]; NULL iff Ln == 0
 *   k_cache, v_cache   : device, [H, capacity, d]  (the rank's head-sharded cache, as in a3)
 *   lse                : device, float [H, Lq] (local head index), or NULL
 *   Everything else as ws_block_causal_attn; workspace size = ..._workspace_bytes(Lq, H, d, ...).
 *   Errors: as a3, plus INVALID_ARG if head_begin < 0 or head_begin + H > H_total.
 * ---------------------------------------------------------------------------------------------- */
int ws_block_causal_attn_seq_layout(void* out_seq, float* lse, const void* q_seq, const void* k_cache,
                                    const void* v_cache, int64_t capacity, int64_t cache_len, const void* k_new_seq,
                                    const void* v_new_seq, int32_t Ln, int32_t H_total, int32_t head_begin, int32_t H,
                                    int32_t d, int32_t Lq, const ws_block_mask* mask, float softmax_scale,
                                    void* workspace, size_t workspace_bytes, ws_dtype dt, void* stream);

/* ------------------------------------------------------------------------------------------------
 * FP8 K/V cache ("local shards of the full-history cache")
 *
 *   The cache rows are stored as OCP FP8 E4M3 codes (1 sign, 4 exponent bits with bias 7, 3 mantissa bits, no
 *   infinity, largest finite value 448) with ONE power-of-two scale 2^e per (row, head), e an int8:
 *
 *     amax = max_c |x[c]| over the row's d elements
 *     e    = the smallest integer with 448 * 2^e >= amax, clamped to [-100, 7]      (amax == 0 -> e = -100)
 *     code = round-to-nearest-even(x / 2^e) to E4M3, saturated to +-448 (reached only when e was clamped at 7,
 *            i.e. |x| > 57344)
 *     dequantised value = decode(code) * 2^e, exactly representable in BF16.
 *
 *   ws_kv_cache_write_fp8:  cache8[h, row_offset + r, :], exp[h, row_offset + r] = quantise(src[r, head_begin + h, :])
 *   for K and V; every other byte is untouched.  BF16 sources only.
 *     k_cache8, v_cache8 : device, uint8 [H, capacity, d]      k_exp, v_exp : device, int8 [H, capacity]
 *     k_src, v_src       : device, BF16 [n_rows, H_src, d]
 *   ws_block_causal_attn_fp8kv:  a3 with that cache; q, k_new, v_new, out stay BF16 [L, H, d].  The codes are
 *   expanded to BF16 inside the SM (exactly), so the result is what ws_block_causal_attn returns on the dequantised
 *   cache, up to the order of FP32 summation.  Workspace size as ws_block_causal_attn (WS_DTYPE_BF16).
 *   Sources must be FINITE.  A NaN element is stored as the E4M3 NaN code (0x7f / 0xff) and leaves the exponent and codes of
 *   its own (row, head) group unspecified (other groups are unaffected); ws_block_causal_attn_fp8kv does not decode NaN codes
 *   as NaN but as the finite value +-480 * 2^e, so a NaN written into the FP8 cache does NOT surface in the output the way it
 *   does with the BF16 cache.  +-Inf saturates to +-448 * 2^7.  (Pinned by tests/test_gpu_fp8.py.)
 *   Both: d in {64, 128}; capacity a multiple of 16 and every pointer 16-byte aligned (ALIGNMENT otherwise); the
 *   other errors as their BF16 counterparts.
 * ---------------------------------------------------------------------------------------------- */
int ws_kv_cache_write_fp8(void* k_cache8, void* v_cache8, int8_t* k_exp, int8_t* v_exp, int64_t capacity, int32_t H, int32_t d,
                          const void* k_src, const void* v_src, int32_t n_rows, int32_t H_src, int32_t head_begin,
                          int64_t row_offset, void* stream);

int ws_block_causal_attn_fp8kv(void* out, float* lse, const void* q, const void* k_cache8, const void* v_cache8,
                               const int8_t* k_exp, const int8_t* v_exp, int64_t capacity, int64_t cache_len, const void* k_new,
                               const void* v_new, int32_t Ln, int32_t H, int32_t d, int32_t Lq, const ws_block_mask* mask,
                               float softmax_scale, void* workspace, size_t workspace_bytes, void* stream);

/* ------------------------------------------------------------------------------------------------
 * Ring (sliding-window) K/V cache (SURVEY.md 8(f).4 "cache windowing/eviction for unbounded sessions"
 * "local shards of the full-history cache", PAPER.md:47 one committed unit per 160 ms without end).  The paper gives no
 * eviction rule; reading R19:
 *
 *   The cache is a ring of `capacity` rows per head that keeps the MOST RECENT rows of the session.  Row w of the
 *   session (w = 0, 1, 2, ...) lives in physical row w mod capacity until row w + capacity overwrites it.  After W rows:
 *       cache_len = min(W, capacity),   ring_start = W < capacity ? 0 : W mod capacity      (ws_ring_state, host only)
 *   and cache key j of the attention timeline (oldest first) is physical row (ring_start + j) mod capacity.
 *
 *   ws_kv_cache_write_ring:  cache[h, (write_pos + r) mod capacity, :] = src[r, head_begin + h, :] for K and V, every
 *     other byte untouched; write_pos = rows of the session written before this call.  Arguments as ws_kv_cache_write.
 *     Errors as ws_kv_cache_write, with OUT_OF_RANGE for write_pos < 0 or n_rows > capacity (a call never overwrites
 *     a row it has written itself).  One launch, two when the slice wraps.
 *   ws_block_causal_attn_ring:  ws_block_causal_attn whose cache keys are the window in timeline order; kv_visible
 *     cuts that timeline.  The window is at most two physical runs of the cache tensor, each read in place by TMA
 *     (no linearised copy); ring_start need not be aligned to anything.  ALL `capacity` rows of the cache tensor must hold
 *     finite values (zero-initialise the ring before the session): a 128-row tile that straddles the window's end reads
 *     rows outside it, which are masked out of the softmax but still multiplied by zero.  Arguments, workspace and errors as ws_block_causal_attn, plus OUT_OF_RANGE unless
 *     0 <= ring_start < capacity.  ring_start == 0 is ws_block_causal_attn itself.
 * ---------------------------------------------------------------------------------------------- */
int ws_kv_cache_write_ring(void* k_cache, void* v_cache, int64_t capacity, int32_t H, int32_t d, const void* k_src,
                           const void* v_src, int32_t n_rows, int32_t H_src, int32_t head_begin, int64_t write_pos, ws_dtype dt,
                           void* stream);

int ws_ring_state(int64_t rows_written, int64_t capacity, int64_t* ring_start /* host */, int64_t* cache_len /* host */);

int ws_block_causal_attn_ring(void* out, float* lse, const void* q, const void* k_cache, const void* v_cache, int64_t capacity,
                              int64_t ring_start, int64_t cache_len, const void* k_new, const void* v_new, int32_t Ln, int32_t H,
                              int32_t d, int32_t Lq, const ws_block_mask* mask, float softmax_scale, void* workspace,
                              size_t workspace_bytes, ws_dtype dt, void* stream);

/* ------------------------------------------------------------------------------------------------
 * Ulysses exchange over peer memory ("denoising for the long latent video sequence is split
 * across ranks with Ulysses all-to-all/gather communication.  Audio latents ... are generated without sequence sharding",
 * :65 "Thinker broadcasts performer-compatible K/V slices", :73, :81).  Index maps: DESIGN.md reading R20.
 *
 *   P ranks (<= WS_MAX_PEERS), H heads in all, Hp = H / P per rank.  A unit's sequence is P * Ls sharded (video) tokens
 *   followed by La unsharded (audio) tokens.  Rank r holds X_r [Ls + La, H, d]: its Ls video tokens, then the La audio
 *   tokens (replicated on every rank).  Attention is head-parallel: rank g needs Y_g [P * Ls + La, Hp, d].
 *
 *   "Peer pointers" are device pointers valid in the CALLING process: local memory, or another GPU's memory mapped
 *   through CUDA peer access / IPC / symmetric memory.  The kernels store through them directly (push model), so the
 *   pack (a2), the unpack (a4) and the cache write (a1) ARE the transport: nothing is staged, no collective library
 *   runs on the data path.  The calls are stream-ordered on the caller's stream and do not synchronise ranks: a
 *   receiver must not read until every sender's call has completed (a barrier between the ranks' streams, e.g. one
 *   torch.distributed barrier or a symmetric-memory signal per exchange), and a sender must not overwrite a buffer a
 *   receiver is still reading.  On a single GPU all peers are local buffers and stream order is enough.
 *
 *   ws_ulysses_push_seq_to_head   exchange #1 (all-to-all) for up to 4 tensors (Q, K_new, V_new) in one call, run by rank `rank`:
 *       Y_g[rank * Ls + t, c, :] = X[t, g * Hp + c, :]    for every peer g (stored through peer_dsts[i * P + g])
 *       Y_rank[P * Ls + a, c, :] = X[Ls + a, rank * Hp + c, :]   (the audio rows are replicated: local)
 *     peer_dsts : host array [n_tensors * P] of peer pointers to tensor i's Y_g;   srcs : host array [n_tensors] of X.
 *   ws_block_causal_attn_push_out   a3 with exchange #2 fused into its epilogue, run by rank `rank` on its H (= Hp) heads:
 *     q, k_new, v_new, caches, lse, mask, workspace exactly as ws_block_causal_attn with Lq = P * Ls + La; the output
 *     row i of head c is stored to
 *       Z_r[t, rank * H + c, :],      r = i / Ls, t = i % Ls          for i <  P * Ls   (all-to-all)
 *       Z_r[Ls + (i - P * Ls), rank * H + c, :]  for EVERY r          for i >= P * Ls   (all-gather of the audio rows)
 *     peer_outs : host array [P] of peer pointers to Z_r [Ls + La, P * H, d]; other heads of Z_r are not touched.
 *   ws_kv_slice_broadcast_write   a1 on every rank by one kernel (the thinker's broadcast fused with the cache write):
 *       cache_g[h, row_offset + i, :] = src[i, g * Hp + h, :]       peer_k_caches / peer_v_caches : host arrays [P]
 *   Errors: as a2 / a3 / a1, plus UNSUPPORTED for P > WS_MAX_PEERS, INVALID_ARG for a NULL peer pointer or rank outside
 *   [0, P), OUT_OF_RANGE if P * Ls > Lq, OVERLAP if two destinations (or a destination and a source) intersect.
 * ---------------------------------------------------------------------------------------------- */
int ws_ulysses_push_seq_to_head(void* const* peer_dsts, const void* const* srcs, int32_t n_tensors, int64_t Ls, int64_t La,
                                int32_t H, int32_t d, int32_t P, int32_t rank, ws_dtype dt, void* stream);

int ws_block_causal_attn_push_out(void* const* peer_outs, int32_t P, int32_t rank, int64_t Ls, float* lse, const void* q,
                                  const void* k_cache, const void* v_cache, int64_t capacity, int64_t cache_len, const void* k_new,
                                  const void* v_new, int32_t Ln, int32_t H, int32_t d, int32_t Lq, const ws_block_mask* mask,
                                  float softmax_scale, void* workspace, size_t workspace_bytes, ws_dtype dt, void* stream);

int ws_kv_slice_broadcast_write(void* const* peer_k_caches, void* const* peer_v_caches, int32_t P, int64_t capacity, int32_t Hp,
                                int32_t d, const void* k_src, const void* v_src, int32_t n_rows, int64_t row_offset, ws_dtype dt,
                                void* stream);

/* ------------------------------------------------------------------------------------------------
 * a5. One unit end to end from HOST buffers ("receive the current K/V slice, update
 *     their local shards of the full-history cache, and run ... denoising for the next unit").
 *
 *   Stream-ordered on `stream`:  H2D copies of the slice and of every step's Q/K_new/V_new ->
 *   ws_kv_cache_write (if n_slice_rows > 0) -> n_steps x attention (step s uses q_host[s],
 *   k_new_host[s], v_new_host[s]; the mask is the single block "all Lq rows see
 *   cache_len_after + Ln keys") -> D2H copy of every step's output into out_host[s].
 *   The unit is PCIe-bound (config 3: 50.8 MB in, 9.9 MB out against 0.27 ms of kernels), so every transfer is one
 *   contiguous cudaMemcpyAsync on an internal copy stream, ordered  slice | Q[s] | K_new[s], V_new[s] | ...,  and the
 *   attention of a step is split by key source: Q[s] against the CACHE starts as soon as the slice and Q[s] have landed
 *   and runs under the transfer of the unit's own K/V; Q[s] against the unit's own rows follows, and a small kernel
 *   merges the two (attention over a union of key sets = LSE-weighted mean of the two attentions; both partial results
 *   stay FP32 until they are merged, so the output is rounded to BF16 once, like ws_block_causal_attn's).  Outputs return on a
 *   second internal stream.  Both helper streams (one pair per device, created on first use: the library's only lazily
 *   created global state besides the driver entry point) start after the work already queued on `stream` and are
 *   joined back into it -- also when a CUDA call fails half way -- so to the caller the call is ordered on `stream`
 *   like any other and a stream capture is never left unjoined.  Calls on the same device from several host threads
 *   are serialised for the length of the enqueue.
 *   The call does not synchronise; the caller synchronises the stream before reading out_host.
 *
 *   k_cache, v_cache : device [H, capacity, d]      (the persistent local cache)
 *   k_slice_host, v_slice_host : host (pinned for async copies) [n_slice_rows, H, d], written at
 *                      row_offset; cache_len_after = valid rows once the slice is in
 *   q_host, k_new_host, v_new_host : host [n_steps][Lq | Ln, H, d] contiguous over steps
 *   out_host         : host [n_steps][Lq, H, d]
 *   staging          : device scratch >= ws_unit_forward_host_staging_bytes(...) (inputs, outputs, the two
 *                      partial results, attention workspace), 256-byte aligned
 *   BF16 only.  Same error rules as the calls it is made of.
 * ---------------------------------------------------------------------------------------------- */
size_t ws_unit_forward_host_staging_bytes(int32_t Lq, int32_t Ln, int32_t H, int32_t d, int32_t n_slice_rows,
                                          int64_t kv_total, int32_t n_steps);

int ws_unit_forward_host(void* out_host, const void* q_host, const void* k_new_host, const void* v_new_host,
                         int32_t Lq, int32_t Ln, int32_t n_steps, void* k_cache, void* v_cache, int64_t capacity,
                         const void* k_slice_host, const void* v_slice_host, int32_t n_slice_rows, int64_t row_offset,
                         int64_t cache_len_after, int32_t H, int32_t d, float softmax_scale, void* staging,
                         size_t staging_bytes, void* stream);

/* Host-only diagnostic (touches no device): the work schedule ws_block_causal_attn would use for this problem on
 * a device with n_sms SMs ("Schedule").  The Q rows of a head are cut into 128-row tiles; tiles
 * (2u, 2u + 1) form PAIR unit u, which runs one iteration per KV tile (unit_kv_tiles[u] of them: what the later
 * tile's last row sees), both tiles on the same KV tile; an odd last tile is a SINGLE unit whose unit_kv_tiles[u]
 * KV tiles are walked two per iteration (unit_iters[u] = ceil(unit_kv_tiles[u] / 2)).  Work item i =
 * head * n_units + unit, n_units = ceil(Lq / 256).  CTA c < *grid runs the whole items w * grid + c for
 * w < *n_waves, then the flattened iterations [pool_begin[c], pool_begin[c + 1]) of the remaining items
 * (coordinate of item i, iteration k: (i / n_units) * sum(unit_iters) + sum(unit_iters[0 .. i % n_units)) + k).
 * Iterations [i0, i1) of a single unit cover its KV tiles [2 i0, min(2 i1, unit_kv_tiles)).
 *   unit_iters, unit_kv_tiles : host, >= ceil(Lq / 256) entries (written);  pool_begin : host, >= n_sms + 1 entries
 * Errors: INVALID_ARG, OUT_OF_RANGE, UNSUPPORTED as for the mask of ws_block_causal_attn. */
int ws_attn_schedule(int32_t Lq, int32_t H, int64_t cache_len, int32_t Ln, const ws_block_mask* mask, int32_t n_sms,
                     int32_t* grid, int32_t* n_waves, int32_t* unit_iters, int32_t* unit_kv_tiles, int64_t* pool_begin);

/* ---- utilities ---- */
const char* ws_status_string(int status); /* static string, never NULL */
int ws_version(void);                     /* WS_VERSION of the loaded library */
int ws_last_cuda_error(void);             /* cudaError_t of the last WS_ERR_CUDA on this thread, else 0 */
int ws_kernel_launch_count(void);         /* kernels this library has launched in this process so far */

#ifdef __cplusplus
}
#endif
#endif /* WS_H_ */
