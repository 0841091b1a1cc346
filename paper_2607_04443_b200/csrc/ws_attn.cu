// ws_attn.cu -- block-causal unit attention for sm_100a (include/ws.h a3).
//
// Flash-style forward pass written directly on the Blackwell primitives:
//   * K/V tiles (128 keys x d) and the two 128-row Q tiles of a CTA are staged in shared memory
//     by TMA (cp.async.bulk.tensor, 128-byte swizzle) through a 5-slot mbarrier ring;
//   * S = Q K^T and O += P V run on the 5th-gen tensor cores (tcgen05.mma, BF16 in, FP32
//     accumulate) with S, P and O living in TMEM: S0,S1 (128 columns each), O0,O1 (d columns
//     each); P overwrites S in place as packed BF16 and is fed back as the TMEM A operand;
//   * the online softmax is done by two 128-thread warpgroups, one per Q tile, one thread per
//     query row (tcgen05.ld 32x32b gives each thread its row: no shuffles), exp2 with the scale
//     folded in, and a lazy rescale of O (only when the running max grows by more than 2^8);
//   * block-causality is exploited at tile level: a unit of work only visits the KV tiles its
//     last row can see, and only boundary tiles pay for per-row column masking;
//   * a CTA has two tile slots (S/P/O sets in TMEM, one softmax warpgroup each) that ping-pong on the
//     tensor pipe.  A work unit is either a PAIR of consecutive 128-row Q tiles of one head (both slots
//     walk the same KV tiles and share each K/V tile in shared memory) or, for the ragged last Q tile of
//     a head, a SINGLE tile whose KV range is cut in two halves, one per slot (the two partial results
//     are merged inside the CTA through TMEM), so a tail tile costs half a pair instead of a whole one;
//   * a persistent stream-K schedule splits the flattened (head, unit, iteration) space evenly over
//     one CTA per SM; a segment that does not cover its unit's whole KV range writes FP32 partials
//     (O, m, l) and a small combine kernel merges them.
//
// Roofline: tensor pipe.  Algorithmic flops = 4 * d * H * sum_b |block b| * kv_visible[b].
#include <cuda.h>
#include <cuda_bf16.h>
#include <cudaTypedefs.h>

#include <cstring>
#include <mutex>
#include <type_traits>

#include "ws_internal.h"
#include "ws_ptx.cuh"

namespace {

constexpr int kBlockM = 128;  // query rows per tile (one TMEM lane each)
constexpr int kBlockN = 128;  // keys per tile
constexpr int kPairM = 2 * kBlockM;
constexpr int kMaxStages = 5; // K/V ring slots (BF16 cache: 5; FP8 cache: 3 + a four-slot staging ring of raw FP8 tiles)
constexpr int kStg = 4;       // FP8 staging slots: the raw tiles are half the size, so the prefetch depth in tiles stays the same
// P is handed to the MMA warp in chunks; chunk c covers the 16-key units [chunk16(c), chunk16(c + 1)) of the tile.
// WS_CHUNK_ENDS lists the chunk ends as decimal digits (2468 = four chunks of 32 keys; 478 = 64 + 48 + 16 keys; the last digit is 8).
// A small LAST chunk shortens what follows the final hand-off on the critical path (its P.V, then the next Q.K^T).
#ifndef WS_CHUNK_ENDS
#define WS_CHUNK_ENDS 478
#endif
__host__ __device__ constexpr int chunk_count() {
  int n = 0;
  for (int v = WS_CHUNK_ENDS; v > 0; v /= 10) ++n;
  return n;
}
constexpr int kPChunks = chunk_count();
__host__ __device__ constexpr int chunk16(int c) {  // first 16-key unit of chunk c; chunk16(kPChunks) == 8
  if (c == 0) return 0;
  int v = WS_CHUNK_ENDS;
  for (int i = kPChunks; i > c; --i) v /= 10;
  return v % 10;
}
// index of the chunk that ends after 16-key unit u (u = 1..8), or -1
__host__ __device__ constexpr int chunk_ending_at(int u) {
  for (int c = 1; c <= kPChunks; ++c)
    if (chunk16(c) == u) return c - 1;
  return -1;
}
static_assert(chunk16(0) == 0 && chunk16(kPChunks) == 8, "chunks cover the 128 keys of a tile");
constexpr int kThreads = 384;  // warp 0 TMA, warp 1 MMA, warp 2 TMEM alloc, warp 3 idle, warps 4-7 / 8-11 softmax
constexpr int kThreads8 = 512; // FP8 cache: a fourth warpgroup (warps 12-15, one per SM sub-partition) turns the raw FP8 tiles into BF16 operand tiles
constexpr int kMaxUnits = 256;  // work units (Q-tile pairs, plus one single tile) per head
constexpr int kMaxCtas = 256; // upper bound on the persistent grid (workspace sizing)
constexpr int kTmemCols = 512;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kRescaleThreshold = 8.0f;  // log2 units: P stays below 2^8
// Which exponentials run on the FMA pipe (degree-3 polynomial) instead of MUFU: bit (u & 1) * 8 + i of the mask selects pair i
// (2 keys) of the 16-key unit u.  0x4949 = pairs 0, 3 and 6 of every unit = 3 exponentials in 8.  Measured on B200 (cfg3,
// profiles/r02b_attn_variants.md): the share has a flat optimum between 1/8 and 3/8, but the POSITIONS matter as much as the
// share (they decide how ptxas interleaves the MUFU and FMA chains): 0x4949 is 1.5 % faster than 0x1111 (1 in 4), another
// 3-in-8 pattern (0x2592) is no better than 0x1111, 1 in 2 (0x5555) is 4 % slower.
#ifndef WS_POLY_MASK
#define WS_POLY_MASK 0x4949
#endif
constexpr unsigned kPolyMask = WS_POLY_MASK;
#ifndef WS_WARP_ARRIVE
#define WS_WARP_ARRIVE 0
#endif
constexpr int kPReadyArrivals = WS_WARP_ARRIVE ? 4 : 128;  // arrivals per P-chunk barrier: one per softmax warp, or one per thread

struct alignas(64) Params {
  CUtensorMap map_q, map_kn, map_vn, map_kc, map_vc;
  // Output rows.  Plain call: n_peers == 1, out_peer[0] = the [Lq, *, d] output.  ws_block_causal_attn_push_out (exchange #2 of
  // the Ulysses group fused into the epilogue): row i < n_peers * peer_rows goes to peer i / peer_rows, local row i % peer_rows;
  // the unsharded rows behind them go to EVERY peer at local row peer_rows + (i - n_peers * peer_rows).  The pointers
  // already carry the offset of this rank's first head.
  void* out_peer[WS_MAX_PEERS];
  int32_t n_peers, peer_rows;
  float* lse;
  float* part_o;   // [records][d/4][128][4]
  float2* part_ml; // [records][128] (m * scale * log2e, l)
  const int8_t* k_exp;  // FP8 cache only: int8 [H, capacity] power-of-two scale exponents of the cache rows
  const int8_t* v_exp;
  int64_t capacity;
  int64_t cache_len;
  // Ring cache (ws_block_causal_attn_ring): cache key j of the timeline is physical row (ring_start + j) mod capacity.  The
  // window is at most two physical runs: A = rows [ring_start, ring_start + len_a) (n_tiles_a KV tiles; the last one may be
  // partial: TMA zero-fills past the tensor's end) and B = rows [0, cache_len - len_a).  Linear cache: ring_start = 0,
  // len_a = cache_len, n_tiles_a = n_cache_tiles.
  int64_t ring_start, len_a;
  int32_t n_tiles_a;
  int64_t out_pitch;  // elements between consecutive tokens of `out` (H * d, or H_total * d for the token-major rank view)
  int32_t Lq, H, Ln, n_blocks, n_units, n_cache_tiles;
  // the last unit of a head is a single Q tile (odd number of Q tiles) that sees last_kv_tiles KV tiles
  int32_t last_single, last_kv_tiles;
  float scale, scale_log2;
  int32_t q_block_end[WS_MAX_MASK_BLOCKS];
  int32_t kv_visible[WS_MAX_MASK_BLOCKS];
  // unit_prefix[u]: CTA iterations before unit u (per head); host-built.  A pair unit takes one iteration per KV
  // tile its later Q tile can see; a single unit takes one iteration per TWO KV tiles (one per slot).
  int32_t unit_prefix[kMaxUnits + 1];
  // Two-phase schedule (host-built).  Work item i = head * n_units + unit.  Phase 1: CTA c runs the whole
  // items w * grid + c, w < n_waves (no partials; the units of one head start together on neighbouring
  // CTAs, so a K/V tile is fetched from DRAM once and hit in L2 by the others).  Phase 2: the
  // remaining items [n_waves * grid, H * n_units) are split stream-K style, CTA c taking the flattened
  // iterations [pool_begin[c], pool_begin[c + 1]) (global coordinates head * Tp + unit_prefix).
  int32_t n_waves, grid;
  int32_t combine_items;  // pool items the combine kernel has work for: split over several CTAs, or without any visible key (0: not launched)
  int32_t combine_max_rec;  // most partial records any of them has per output row
  int64_t pool_begin[kMaxCtas + 1];
};

// ---------------------------------------------------------------------------------------------
// schedule helpers (shared by the attention and the combine kernel)
// ---------------------------------------------------------------------------------------------
// The block tables are read straight from the __grid_constant__ parameter block (constant bank).
__device__ __forceinline__ int block_of_row(const Params& p, int row) {
  int lo = 0, hi = p.n_blocks - 1;  // first b with row < q_block_end[b]
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (row < p.q_block_end[mid]) hi = mid; else lo = mid + 1;
  }
  return lo;
}

// Where output row `row` goes: destinations out_peer[peer0 .. peer0 + n_dst), each at element offset elem_off (to which the
// caller adds head * D + column).
struct RowDst {
  int peer0, n_dst;
  int64_t elem_off;
};
__device__ __forceinline__ RowDst row_dst(const Params& p, int row) {
  RowDst r;
  r.peer0 = 0;
  r.n_dst = 1;
  int64_t local = row;
  if (p.n_peers > 1) {
    const int sharded = p.n_peers * p.peer_rows;
    if (row < sharded) {
      r.peer0 = row / p.peer_rows;
      local = row - r.peer0 * p.peer_rows;
    } else {
      r.n_dst = p.n_peers;
      local = p.peer_rows + (row - sharded);
    }
  }
  r.elem_off = local * p.out_pitch;
  return r;
}

__device__ __forceinline__ int unit_of_iter(const Params& s, int rem) {
  int lo = 0, hi = s.n_units - 1;  // largest u with unit_prefix[u] <= rem
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (s.unit_prefix[mid] <= rem) lo = mid; else hi = mid - 1;
  }
  return lo;
}

// the CTA whose phase-2 range holds flattened iteration t (pool_begin is non-decreasing; empty ranges are skipped)
__device__ __forceinline__ int cta_of_iter(const Params& p, int64_t t) {
  int lo = 0, hi = p.grid - 1;  // largest c with pool_begin[c] <= t
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (p.pool_begin[mid] <= t) lo = mid; else hi = mid - 1;
  }
  return lo;
}

// CTA c takes no pool iteration: the cost-aware partition leaves a CTA empty when its phase-1 items were the expensive
// ones.  Such a CTA may sit INSIDE the CTA span of a split item; it writes no partial record.
__device__ __forceinline__ bool pool_empty(const Params& p, int c) { return p.pool_begin[c] == p.pool_begin[c + 1]; }

struct Segment {
  int head, unit, i0, i1, n_iters;  // iterations [i0, i1) of the unit's n_iters
};

// Walks the CTA's phase-2 share [t, hi) of the flattened iteration space.
__device__ __forceinline__ Segment next_pool_segment(const Params& p, int64_t& t, int64_t hi) {
  const int Tp = p.unit_prefix[p.n_units];
  Segment g;
  g.head = (int)(t / Tp);
  const int rem = (int)(t - (int64_t)g.head * Tp);
  g.unit = unit_of_iter(p, rem);
  g.n_iters = p.unit_prefix[g.unit + 1] - p.unit_prefix[g.unit];
  g.i0 = rem - p.unit_prefix[g.unit];
  const int64_t left = hi - t;
  g.i1 = (int)min((int64_t)g.n_iters, g.i0 + left);
  t += g.i1 - g.i0;
  return g;
}

// A CTA's walk over its segments: whole items first (phase 1), then its stream-K range (phase 2).
// Every role of the CTA runs the same walk, so they agree on the segment sequence.  A unit that
// sees no key at all is reported with n_iters == 0 (phase 1 only): the softmax warps zero-fill its
// rows, the TMA and MMA warps skip it.
struct SegWalk {
  int wave;
  int64_t t, hi;
  __device__ __forceinline__ SegWalk(const Params& p) : wave(0), t(p.pool_begin[blockIdx.x]), hi(p.pool_begin[blockIdx.x + 1]) {}
  __device__ __forceinline__ bool next(const Params& p, Segment& g) {
    if (wave < p.n_waves) {
      const int item = wave * p.grid + (int)blockIdx.x;
      ++wave;
      g.head = item / p.n_units;
      g.unit = item - g.head * p.n_units;
      g.n_iters = p.unit_prefix[g.unit + 1] - p.unit_prefix[g.unit];
      g.i0 = 0;
      g.i1 = g.n_iters;
      return true;
    }
    if (t < hi) {
      g = next_pool_segment(p, t, hi);
      return true;
    }
    return false;
  }
};

// What the two tile slots of the CTA do in a segment.  Slot s runs Q tile q_tile[s] against the KV tiles
// jb[s], jb[s] + 1, ... for n_it iterations.  Pair: both slots walk the same KV tiles (shared K/V tiles in shared
// memory).  Single: the segment's KV tiles [2 i0, min(2 i1, n)) are cut in two runs of n_it tiles; a run that
// reaches past the visible range computes fully masked tiles (TMA zero fill beyond the tensors), which contribute
// nothing.
struct SlotPlan {
  int q_tile[2], jb[2], n_it;
  bool single, whole;  // whole: the segment covers the unit's entire KV range
};
__device__ __forceinline__ SlotPlan plan_of(const Params& p, const Segment& g) {
  SlotPlan sp;
  sp.single = p.last_single && g.unit == p.n_units - 1;
  sp.whole = g.i0 == 0 && g.i1 == g.n_iters;
  sp.n_it = g.i1 - g.i0;
  sp.q_tile[0] = 2 * g.unit;
  if (sp.single) {
    sp.q_tile[1] = 2 * g.unit;
    sp.jb[0] = 2 * g.i0;
    sp.jb[1] = 2 * g.i0 + sp.n_it;
  } else {
    sp.q_tile[1] = 2 * g.unit + 1;
    sp.jb[0] = sp.jb[1] = g.i0;
  }
  return sp;
}

// ---------------------------------------------------------------------------------------------
// the attention kernel
// ---------------------------------------------------------------------------------------------
template <int D, bool KV8 = false>
struct Cfg {
  static constexpr int kStages = KV8 ? 3 : 5;             // BF16 operand ring
  static constexpr int kAtoms = D / 64;                   // 64-element (128-byte) swizzle atoms along d
  static constexpr int kAtomBytes = kBlockN * 128;        // [128 rows][128 B]
  static constexpr int kTileBytes = kAtoms * kAtomBytes;  // one Q tile == one K or V tile
  static constexpr int kSmemQ = 2 * kTileBytes;
  static constexpr int kSmemKV = kStages * kTileBytes;
  static constexpr int kRawTileBytes = kBlockN * D;       // FP8 tile: [128 rows][D bytes], row-major, no swizzle
  static constexpr int kRawSlotBytes = kRawTileBytes + 256;  // + the 128 scale exponents of its rows
  static constexpr int kSmemRaw = KV8 ? kStg * kRawSlotBytes : 0;
  static constexpr int kSmemMerge = kBlockM * 8;           // (m, l) of slot 1 for the in-CTA merge of a single unit
  static constexpr int kSmemBytes = kSmemQ + kSmemKV + kSmemRaw + 256 /*barriers*/ + kSmemMerge;
  static_assert(kSmemBytes <= 227 * 1024, "shared memory budget");
  static constexpr int kThreadsCta = KV8 ? kThreads8 : kThreads;
  static constexpr uint32_t kTmemS0 = 0, kTmemS1 = 128, kTmemO0 = 256, kTmemO1 = 256 + D;
  static constexpr uint32_t kIdescQK = ptx::make_idesc_bf16(kBlockM, kBlockN, false);
  static constexpr uint32_t kIdescPV = ptx::make_idesc_bf16(kBlockM, D, true);
};

struct Barriers {
  uint64_t kv_full[kMaxStages], kv_empty[kMaxStages];
  uint64_t raw_full[kStg], raw_empty[kStg];  // FP8 cache: TMA -> conversion warps
  uint64_t q_full, q_empty;
  uint64_t s_full[2], p_ready[2][kPChunks], o_done[2];  // p_ready[t][c]: chunk c of tile t's P is in TMEM
  uint32_t tmem_base;
};

template <int D, bool OUT_F32, bool KV8>
__global__ void __launch_bounds__(KV8 ? kThreads8 : kThreads, 1) attn_fwd_kernel(const __grid_constant__ Params p) {
  using C = Cfg<D, KV8>;
  constexpr int kStages = C::kStages;
  // 1024-byte alignment is required by the 128-byte swizzle (TMA box and UMMA descriptor agree on it)
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t smem_base = ptx::smem_u32(smem_raw);
  if ((smem_base & 1023u) != 0) __trap();
  uint8_t* smem = smem_raw;
  const uint32_t sQ = smem_base;
  const uint32_t sKV = smem_base + C::kSmemQ;
  const uint32_t sRaw = smem_base + C::kSmemQ + C::kSmemKV;
  Barriers& bar = *reinterpret_cast<Barriers*>(smem + C::kSmemQ + C::kSmemKV + C::kSmemRaw);
  static_assert(sizeof(Barriers) <= 256, "barrier block");
  float2* merge_ml = reinterpret_cast<float2*>(smem + C::kSmemQ + C::kSmemKV + C::kSmemRaw + 256);

  // the warp index goes through a shuffle so that ptxas knows it is warp-uniform: the TMA and MMA
  // warps then run in uniform control flow and their descriptors live in uniform registers
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int i = 0; i < kStages; ++i) {
      // FP8 cache: every operand tile is handed to the MMA warp by the 128 conversion threads
      ptx::mbar_init(ptx::smem_u32(&bar.kv_full[i]), KV8 ? 4 * 32 : 1);
      ptx::mbar_init(ptx::smem_u32(&bar.kv_empty[i]), 1);
    }
    if constexpr (KV8) {
      for (int i = 0; i < kStg; ++i) {
        ptx::mbar_init(ptx::smem_u32(&bar.raw_full[i]), 1);
        ptx::mbar_init(ptx::smem_u32(&bar.raw_empty[i]), 4 * 32);
      }
    }
    ptx::mbar_init(ptx::smem_u32(&bar.q_full), 1);
    ptx::mbar_init(ptx::smem_u32(&bar.q_empty), 1);
    for (int t = 0; t < 2; ++t) {
      ptx::mbar_init(ptx::smem_u32(&bar.s_full[t]), 1);
      for (int c = 0; c < kPChunks; ++c) ptx::mbar_init(ptx::smem_u32(&bar.p_ready[t][c]), kPReadyArrivals);
      ptx::mbar_init(ptx::smem_u32(&bar.o_done[t]), 1);
    }
    ptx::fence_mbar_init();
    ptx::prefetch_tensormap(&p.map_q);
    ptx::prefetch_tensormap(&p.map_kc);
    ptx::prefetch_tensormap(&p.map_vc);
    ptx::prefetch_tensormap(&p.map_kn);
    ptx::prefetch_tensormap(&p.map_vn);
  }
  if (warp == 2) {
    ptx::tmem_alloc(ptx::smem_u32(&bar.tmem_base), kTmemCols);
    ptx::tmem_relinquish();
  }
  __syncthreads();
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem = bar.tmem_base;
  // everything above touched only shared memory, TMEM and the kernel parameters: it overlaps the previous kernel's tail
  wsi::pdl_trigger();
  wsi::pdl_wait();

  if (warp < 4 || warp >= 12) {
    // register budget per warpgroup (FP8 cache: 512 threads x 128 at launch): TMA / MMA 56, conversion 56, softmax 2 x 200
    // (softmax spills below 200; 88 registers and four loads in flight for the conversion warps measured slower for it)
    ptx::setmaxnreg_dec<56>();
    // Both single-issuer roles run on a WHOLE warp in uniform control flow (every lane walks the
    // schedule and waits on the barriers); only the TMA / tcgen05 instructions themselves sit under
    // elect.sync.  A lone `lane == 0` thread would force ptxas to wrap every UTCHMMA / UTMALDG in a
    // register->uniform-register waterfall loop (measured: ~100 cycles of issue per MMA).
    auto bcast_segment = [&](Segment g) {
      g.head = __shfl_sync(0xffffffffu, g.head, 0);
      g.unit = __shfl_sync(0xffffffffu, g.unit, 0);
      g.i0 = __shfl_sync(0xffffffffu, g.i0, 0);
      g.i1 = __shfl_sync(0xffffffffu, g.i1, 0);
      g.n_iters = __shfl_sync(0xffffffffu, g.n_iters, 0);
      return g;
    };
    const int n_cache_tiles = p.n_cache_tiles;
    if (warp == 0) {
      // ============================== TMA producer ==============================
      // Ring order per segment: K of iteration 0 (one tile, or one per slot when the slots walk different KV
      // tiles), then per iteration V (one or two), K of the next iteration (one or two).
      uint32_t it = 0, seg = 0;
      auto load_kv = [&](int head, int j, bool is_v) {
        const uint32_t slot = it % kStages, ph = (it / kStages) & 1;
        const uint32_t dst = sKV + slot * C::kTileBytes;
        const bool from_cache = j < n_cache_tiles;
        uint32_t full;
        if constexpr (KV8) {
          // FP8 cache: this warp only streams the raw cache tiles into the staging ring (counter it = staging uses); the
          // operand ring belongs to the conversion warps, which also fetch the tiles of the unit's own BF16 rows --
          // a second agent claiming ring slots out of order could not tell ring phases apart by parity
          if (!from_cache) return;
          const uint32_t st = it % kStg;
          ptx::mbar_wait(ptx::smem_u32(&bar.raw_empty[st]), ((it / kStg) & 1) ^ 1);
          full = ptx::smem_u32(&bar.raw_full[st]);
          const uint32_t raw = sRaw + st * C::kRawSlotBytes;
          const int64_t rows_left = p.capacity - (int64_t)j * kBlockN;
          const uint32_t n_exp = (uint32_t)(rows_left < kBlockN ? rows_left : kBlockN);  // capacity is a multiple of 16
          if (ptx::elect_one()) {
            ptx::mbar_arrive_expect_tx(full, C::kRawTileBytes + n_exp);
            ptx::tma_load_3d(raw, is_v ? (const void*)&p.map_vc : (const void*)&p.map_kc, full, 0, j * kBlockN, head);
            ptx::bulk_load(raw + C::kRawTileBytes, (is_v ? p.v_exp : p.k_exp) + (int64_t)head * p.capacity + (int64_t)j * kBlockN, n_exp, full);
          }
          __syncwarp();
          ++it;
          return;
        } else {
          ptx::mbar_wait(ptx::smem_u32(&bar.kv_empty[slot]), ph ^ 1);
          full = ptx::smem_u32(&bar.kv_full[slot]);
        }
        if (ptx::elect_one()) {
          ptx::mbar_arrive_expect_tx(full, C::kTileBytes);
          if (from_cache) {
            const void* map = is_v ? (const void*)&p.map_vc : (const void*)&p.map_kc;
            const int r0 = j < p.n_tiles_a ? (int)p.ring_start + j * kBlockN : (j - p.n_tiles_a) * kBlockN;  // run A / run B of a ring
#pragma unroll
            for (int a = 0; a < C::kAtoms; ++a) ptx::tma_load_3d(dst + a * C::kAtomBytes, map, full, a * 64, r0, head);
          } else {
            const void* map = is_v ? (const void*)&p.map_vn : (const void*)&p.map_kn;
            const int r0 = (j - n_cache_tiles) * kBlockN;
#pragma unroll
            for (int a = 0; a < C::kAtoms; ++a) ptx::tma_load_3d(dst + a * C::kAtomBytes, map, full, a * 64, head, r0);
          }
        }
        __syncwarp();
        ++it;
      };
      SegWalk walk(p);
      for (Segment g0; walk.next(p, g0);) {
        const Segment g = bcast_segment(g0);
        const SlotPlan sp = plan_of(p, g);
        if (sp.n_it == 0) continue;
        ptx::mbar_wait(ptx::smem_u32(&bar.q_empty), (seg & 1) ^ 1);
        const uint32_t qf = ptx::smem_u32(&bar.q_full);
        if (ptx::elect_one()) {
          const int n_q = sp.single ? 1 : 2;  // a single unit keeps its one Q tile in Q slot 0 for both tile slots
          ptx::mbar_arrive_expect_tx(qf, n_q * C::kTileBytes);
          for (int tile = 0; tile < n_q; ++tile)
#pragma unroll
            for (int a = 0; a < C::kAtoms; ++a)
              ptx::tma_load_3d(sQ + tile * C::kTileBytes + a * C::kAtomBytes, &p.map_q, qf, a * 64, g.head,
                               (sp.q_tile[0] + tile) * kBlockM);
        }
        __syncwarp();
        load_kv(g.head, sp.jb[0], false);
        if (sp.single) load_kv(g.head, sp.jb[1], false);
        for (int k = 0; k < sp.n_it; ++k) {
          load_kv(g.head, sp.jb[0] + k, true);
          if (sp.single) load_kv(g.head, sp.jb[1] + k, true);
          if (k + 1 < sp.n_it) {
            load_kv(g.head, sp.jb[0] + k + 1, false);
            if (sp.single) load_kv(g.head, sp.jb[1] + k + 1, false);
          }
        }
        ++seg;
      }
    } else if (warp == 1) {
      // ============================== MMA issuer ==============================
      uint32_t it = 0, seg = 0, p_phase = 0;
      const uint32_t tmem_u = __shfl_sync(0xffffffffu, tmem, 0);
      // K-major SW128 operand (Q, K): LBO 16 B, SBO 1024 B; MN-major SW128 operand (V): LBO = atom, SBO 1024 B
      constexpr uint64_t kDescK = ((uint64_t)(16 >> 4) << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
      constexpr uint64_t kDescV = ((uint64_t)(C::kAtomBytes >> 4) << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
      const uint64_t dQ = kDescK | (uint64_t)((sQ & 0x3FFFFu) >> 4);
      const uint64_t dKV = (uint64_t)((sKV & 0x3FFFFu) >> 4);
      // S(tile) = Q(q_slot) . K(slot)^T
      auto issue_qk = [&](int tile, int q_slot, uint32_t slot) {
        const uint64_t qa = dQ + (uint64_t)(q_slot * (C::kTileBytes >> 4));
        const uint64_t kb = (kDescK | dKV) + (uint64_t)(slot * (C::kTileBytes >> 4));
        const uint32_t ts = tmem_u + (tile ? C::kTmemS1 : C::kTmemS0);
#pragma unroll
        for (int k = 0; k < D / 16; ++k) {
          const uint32_t off = ((k >> 2) * C::kAtomBytes + (k & 3) * 32) >> 4;
          ptx::mma_ss(ts, qa + off, kb + off, C::kIdescQK, k > 0);
        }
      };
      // O(tile) (+)= P(tile)[:, 16-key units of chunk] . V(slot)[those keys, :]
      auto issue_pv = [&](int tile, uint32_t slot, int chunk, bool acc) {
        const uint64_t vb = (kDescV | dKV) + (uint64_t)(slot * (C::kTileBytes >> 4));
        const uint32_t ts = tmem_u + (tile ? C::kTmemS1 : C::kTmemS0);
        const uint32_t to = tmem_u + (tile ? C::kTmemO1 : C::kTmemO0);
#pragma unroll
        for (int k = chunk16(chunk); k < chunk16(chunk + 1); ++k) {
          ptx::mma_ts(to, ts + k * 8, vb + (uint64_t)(k * (2048 >> 4)), C::kIdescPV, acc || k > 0);
        }
      };
      auto wait_full = [&](uint32_t i) {
        ptx::mbar_wait(ptx::smem_u32(&bar.kv_full[i % kStages]), (i / kStages) & 1);
        ptx::tc_fence_after();
      };
      SegWalk walk(p);
      for (Segment g0; walk.next(p, g0);) {
        const Segment g = bcast_segment(g0);
        const SlotPlan sp = plan_of(p, g);
        if (sp.n_it == 0) continue;
        const bool split = sp.single;     // the slots use separate K/V tiles
        const int q_slot1 = split ? 0 : 1;
        ptx::mbar_wait(ptx::smem_u32(&bar.q_full), seg & 1);
        {
          const uint32_t it_a = it++, it_b = split ? it++ : it_a;
          wait_full(it_a);
          if (ptx::elect_one()) {
            issue_qk(0, 0, it_a % kStages);
            ptx::tc_commit(ptx::smem_u32(&bar.s_full[0]));
            if (split) ptx::tc_commit(ptx::smem_u32(&bar.kv_empty[it_a % kStages]));
          }
          __syncwarp();
          if (split) wait_full(it_b);
          if (ptx::elect_one()) {
            issue_qk(1, q_slot1, it_b % kStages);
            ptx::tc_commit(ptx::smem_u32(&bar.s_full[1]));
            ptx::tc_commit(ptx::smem_u32(&bar.kv_empty[it_b % kStages]));
            if (sp.n_it == 1) ptx::tc_commit(ptx::smem_u32(&bar.q_empty));
          }
          __syncwarp();
        }
        for (int k = 0; k < sp.n_it; ++k) {
          const bool has_next = k + 1 < sp.n_it, acc = k > 0;
          uint32_t it_v[2], it_k[2] = {0, 0};
          it_v[0] = it++;
          it_v[1] = split ? it++ : it_v[0];
          if (has_next) { it_k[0] = it++; it_k[1] = split ? it++ : it_k[0]; }
          wait_full(it_v[0]);
#pragma unroll
          for (int tile = 0; tile < 2; ++tile) {
            const uint32_t slot_v = it_v[tile] % kStages, slot_k = it_k[tile] % kStages;
            if (tile == 1 && split) wait_full(it_v[1]);
#pragma unroll
            for (int c = 0; c + 1 < kPChunks; ++c) {
              ptx::mbar_wait(ptx::smem_u32(&bar.p_ready[tile][c]), p_phase);
              ptx::tc_fence_after();
              if (ptx::elect_one()) issue_pv(tile, slot_v, c, acc);
              __syncwarp();
            }
            ptx::mbar_wait(ptx::smem_u32(&bar.p_ready[tile][kPChunks - 1]), p_phase);
            ptx::tc_fence_after();
            if (has_next && (tile == 0 || split)) wait_full(it_k[tile]);
            if (ptx::elect_one()) {
              issue_pv(tile, slot_v, kPChunks - 1, acc);
              ptx::tc_commit(ptx::smem_u32(&bar.o_done[tile]));
              if (tile == 1 || split) ptx::tc_commit(ptx::smem_u32(&bar.kv_empty[slot_v]));
              if (has_next) {
                issue_qk(tile, tile ? q_slot1 : 0, slot_k);
                ptx::tc_commit(ptx::smem_u32(&bar.s_full[tile]));
                if (tile == 1 || split) ptx::tc_commit(ptx::smem_u32(&bar.kv_empty[slot_k]));
                if (tile == 1 && k + 2 == sp.n_it) ptx::tc_commit(ptx::smem_u32(&bar.q_empty));
              }
            }
            __syncwarp();
          }
          p_phase ^= 1;
        }
        ++seg;
      }
    } else if (KV8 && warp >= 12) {
      // ============================== FP8 -> BF16 conversion warps ==============================
      // Walk the tiles in the TMA producer's order.  A cache tile: raw E4M3 bytes [128 rows][D] plus the rows' scale
      // exponents sit in the staging slot; code b of a row with exponent e becomes the BF16 number
      // decode(b) * 2^e, written into the operand ring in the 128-byte-swizzled layout TMA would have produced.
      // decode: the 7 magnitude bits of b, placed at BF16 bits [10:4], read as a BF16 number give decode(|b|) * 2^-120
      // for normal AND subnormal codes alike, so one BF16 multiply by 2^(120 + e) finishes the job exactly.
      if constexpr (KV8) {
        const int row = (warp - 12) * 32 + lane;  // one thread per tile row
        uint32_t it = 0, it_raw = 0;  // operand-ring uses (every tile), staging uses (cache tiles)
        auto convert = [&](int head, int j, bool is_v) {
          const uint32_t slot = it % kStages;
          const uint32_t full = ptx::smem_u32(&bar.kv_full[slot]);
          ptx::mbar_wait(ptx::smem_u32(&bar.kv_empty[slot]), ((it / kStages) & 1) ^ 1);
          ++it;
          if (j >= n_cache_tiles) {
            // a tile of the unit's own BF16 rows: TMA straight into the ring slot; the issuing thread's arrival carries the bytes
            const uint32_t dstn = sKV + slot * C::kTileBytes;
            if (warp == 12 && ptx::elect_one()) {
              ptx::mbar_arrive_expect_tx(full, C::kTileBytes);
              const void* map = is_v ? (const void*)&p.map_vn : (const void*)&p.map_kn;
              const int r0 = (j - n_cache_tiles) * kBlockN;
#pragma unroll
              for (int a = 0; a < C::kAtoms; ++a) ptx::tma_load_3d(dstn + a * C::kAtomBytes, map, full, a * 64, head, r0);
            } else {
              ptx::mbar_arrive(full);
            }
            __syncwarp();
            return;
          }
          const uint32_t st = it_raw % kStg;
          ptx::mbar_wait(ptx::smem_u32(&bar.raw_full[st]), (it_raw / kStg) & 1);
          ++it_raw;
          {
            const uint32_t raw = sRaw + st * C::kRawSlotBytes + row * D, dst = sKV + slot * C::kTileBytes + row * 128;
            int e = ptx::lds_s8(sRaw + st * C::kRawSlotBytes + C::kRawTileBytes + row);
            e = e < -100 ? -100 : (e > 7 ? 7 : e);  // rows past the cache's end carry stale bytes: keep the factor finite
            const uint32_t mult = (uint32_t)(247 + e) << 7, mult2 = mult | (mult << 16);
            // 16 codes (16 bytes) per step; the threads of a quarter-warp read different 16-byte slots of their rows
            // (row pitch D = 128 or 64 bytes: the same slot of eight consecutive rows would share banks)
            constexpr int kRowsPerLine = 128 / D;
            constexpr int kBatch = 2;  // 16-byte loads in flight per thread (56 registers)
#pragma unroll
            for (int i0 = 0; i0 < D / 16; i0 += kBatch) {
              uint32_t w[kBatch][4];
#pragma unroll
              for (int b = 0; b < kBatch; ++b) ptx::lds128(raw + (((i0 + b) ^ ((row / kRowsPerLine) & (D / 16 - 1))) << 4), w[b]);
#pragma unroll
              for (int b = 0; b < kBatch; ++b) {
                const int c16 = (i0 + b) ^ ((row / kRowsPerLine) & (D / 16 - 1));
                uint32_t o[8];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                  o[2 * k] = ptx::e4m3x2_to_bf16x2_scaled(__byte_perm(w[b][k], 0, 0x1404), mult2);
                  o[2 * k + 1] = ptx::e4m3x2_to_bf16x2_scaled(__byte_perm(w[b][k], 0, 0x3424), mult2);
                }
                // BF16 columns [16 c16, 16 c16 + 16): 16-byte chunks 2 c16 and 2 c16 + 1 of the row, inside atom c16 / 4
                const uint32_t base = dst + (c16 >> 2) * C::kAtomBytes;
                const int ch = (c16 & 3) * 2;
                ptx::sts128(base + (((ch) ^ (row & 7)) << 4), *reinterpret_cast<uint32_t(*)[4]>(&o[0]));
                ptx::sts128(base + (((ch + 1) ^ (row & 7)) << 4), *reinterpret_cast<uint32_t(*)[4]>(&o[4]));
              }
            }
            ptx::fence_proxy_async();  // the tensor core reads shared memory through the async proxy
          }
          ptx::mbar_arrive(full);
          ptx::mbar_arrive(ptx::smem_u32(&bar.raw_empty[st]));
        };
        SegWalk walk(p);
        for (Segment g; walk.next(p, g);) {
          const SlotPlan sp = plan_of(p, g);
          if (sp.n_it == 0) continue;
          convert(g.head, sp.jb[0], false);
          if (sp.single) convert(g.head, sp.jb[1], false);
          for (int k = 0; k < sp.n_it; ++k) {
            convert(g.head, sp.jb[0] + k, true);
            if (sp.single) convert(g.head, sp.jb[1] + k, true);
            if (k + 1 < sp.n_it) {
              convert(g.head, sp.jb[0] + k + 1, false);
              if (sp.single) convert(g.head, sp.jb[1] + k + 1, false);
            }
          }
        }
      }
    }
  } else {
    // ============================== softmax warpgroups ==============================
    ptx::setmaxnreg_inc<KV8 ? 200 : 224>();
    const int tile = (warp - 4) >> 2;                    // 0 or 1: which tile slot of the CTA
    const int row_in_tile = ((warp & 3) << 5) | lane;    // == TMEM lane this thread may access
    const uint32_t lane_off = (uint32_t)((warp & 3) << 5) << 16;
    const uint32_t tS = tmem + (tile ? C::kTmemS1 : C::kTmemS0) + lane_off;
    const uint32_t tO = tmem + (tile ? C::kTmemO1 : C::kTmemO0) + lane_off;
    const uint32_t s_full = ptx::smem_u32(&bar.s_full[tile]);
    const uint32_t p_ready = ptx::smem_u32(&bar.p_ready[tile][0]);
    const uint32_t o_done = ptx::smem_u32(&bar.o_done[tile]);
    uint32_t n_iter = 0;  // S tiles consumed so far == PVs requested so far (drives every phase bit)

    // final rows: O / l in the output dtype, LSE
    auto store_row = [&](int head, int row, float inv, uint32_t t_src, auto&& transform) {
      const RowDst rd = row_dst(p, row);
#pragma unroll
      for (int ch = 0; ch < D / 32; ++ch) {
        uint32_t o[32];
        ptx::tmem_ld32(t_src + ch * 32, o);
        ptx::tc_wait_ld();
        transform(ch, o);
        if (row < p.Lq) {
          const int64_t off = rd.elem_off + (int64_t)head * D + ch * 32;
          if constexpr (OUT_F32) {
            float4 v[8];
#pragma unroll
            for (int c = 0; c < 8; ++c)
              v[c] = make_float4(__uint_as_float(o[4 * c]) * inv, __uint_as_float(o[4 * c + 1]) * inv,
                                 __uint_as_float(o[4 * c + 2]) * inv, __uint_as_float(o[4 * c + 3]) * inv);
            for (int k = 0; k < rd.n_dst; ++k) {
              float4* dst = reinterpret_cast<float4*>(reinterpret_cast<float*>(p.out_peer[rd.peer0 + k]) + off);
#pragma unroll
              for (int c = 0; c < 8; ++c) dst[c] = v[c];
            }
          } else {
            uint4 v[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              v[c].x = ptx::pack_bf16(__uint_as_float(o[8 * c]) * inv, __uint_as_float(o[8 * c + 1]) * inv);
              v[c].y = ptx::pack_bf16(__uint_as_float(o[8 * c + 2]) * inv, __uint_as_float(o[8 * c + 3]) * inv);
              v[c].z = ptx::pack_bf16(__uint_as_float(o[8 * c + 4]) * inv, __uint_as_float(o[8 * c + 5]) * inv);
              v[c].w = ptx::pack_bf16(__uint_as_float(o[8 * c + 6]) * inv, __uint_as_float(o[8 * c + 7]) * inv);
            }
            for (int k = 0; k < rd.n_dst; ++k) {
              uint4* dst = reinterpret_cast<uint4*>(reinterpret_cast<__nv_bfloat16*>(p.out_peer[rd.peer0 + k]) + off);
#pragma unroll
              for (int c = 0; c < 4; ++c) dst[c] = v[c];
            }
          }
        }
      }
    };

    SegWalk walk(p);
    for (Segment g; walk.next(p, g);) {
      const SlotPlan sp = plan_of(p, g);
      const int row = (tile ? sp.q_tile[1] : sp.q_tile[0]) * kBlockM + row_in_tile;
      const bool row_valid = row < p.Lq;
      if (sp.n_it == 0) {
        // no key is visible to this unit (reading R11): output rows 0, LSE -inf (a single unit: slot 0 writes them)
        if (row_valid && !(sp.single && tile == 1)) {
          if (p.lse != nullptr) p.lse[(int64_t)g.head * p.Lq + row] = -INFINITY;
          constexpr int kRowVecs = D * (OUT_F32 ? 4 : 2) / 16;
          const RowDst rd = row_dst(p, row);
          for (int k = 0; k < rd.n_dst; ++k) {
            uint4* dst = reinterpret_cast<uint4*>(reinterpret_cast<char*>(p.out_peer[rd.peer0 + k]) + (rd.elem_off + (int64_t)g.head * D) * (OUT_F32 ? 4 : 2));
#pragma unroll
            for (int c = 0; c < kRowVecs; ++c) dst[c] = make_uint4(0u, 0u, 0u, 0u);
          }
        }
        continue;
      }
      // padding rows (>= Lq; their Q is TMA zero fill, their output is never stored) see what the last real row
      // sees: masking them would push their whole warp onto the slower boundary path for every tile
      const int nvis = p.kv_visible[block_of_row(p, min(row, p.Lq - 1))];
      const int vis_cache = (int)min((int64_t)nvis, p.cache_len);
      const int vis_a = (int)min((int64_t)vis_cache, p.len_a);  // visible rows of the cache's first physical run
      float m = -INFINITY, l = 0.f;  // running max in raw-score units, running sum
      const int j_begin = tile ? sp.jb[1] : sp.jb[0];

      for (int k = 0; k < sp.n_it; ++k, ++n_iter) {
        const int j = j_begin + k;
        int lim;  // columns [0, lim) of this tile are visible to this row (<= 0: none; a run past the visible range)
        if (j < p.n_tiles_a) lim = vis_a - j * kBlockN;
        else if (j < p.n_cache_tiles) lim = vis_cache - (int)p.len_a - (j - p.n_tiles_a) * kBlockN;  // second run of a ring
        else lim = nvis - (int)p.cache_len - (j - p.n_cache_tiles) * kBlockN;

        ptx::mbar_wait(s_full, n_iter & 1);
        ptx::tc_fence_after();
        uint32_t s[4][32];
#pragma unroll
        for (int q = 0; q < 4; ++q) ptx::tmem_ld32(tS + q * 32, s[q]);
        ptx::tc_wait_ld();
        if (lim < kBlockN) {
#pragma unroll
          for (int q = 0; q < 4; ++q)
#pragma unroll
            for (int c = 0; c < 32; ++c)
              if (q * 32 + c >= lim) s[q][c] = 0xff800000u;  // -inf
        }
        // row maximum: 8 independent chains (a single chain is latency-bound: 64 dependent FMNMX3)
        float mx8[8];
#pragma unroll
        for (int a = 0; a < 8; ++a) mx8[a] = __uint_as_float(s[0][a]);
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
          for (int c = (q == 0 ? 8 : 0); c < 32; c += 16)
#pragma unroll
            for (int a = 0; a < 8; ++a)
              mx8[a] = fmaxf(mx8[a], fmaxf(__uint_as_float(s[q][c + a]), __uint_as_float(s[q][(c + 8 + a) & 31])));
        const float mx = fmaxf(fmaxf(fmaxf(mx8[0], mx8[1]), fmaxf(mx8[2], mx8[3])), fmaxf(fmaxf(mx8[4], mx8[5]), fmaxf(mx8[6], mx8[7])));
        const float m_new = fmaxf(m, mx);
        const bool grow = (m_new - m) * p.scale_log2 > kRescaleThreshold;  // false when both are -inf (NaN)
        if (k == 0) {
          m = m_new;  // O is overwritten by the first P.V of the segment: nothing to rescale
        } else if (__any_sync(0xffffffffu, grow)) {
          // lazy rescale of the accumulator in TMEM: needs the previous P.V to have landed
          ptx::mbar_wait(o_done, (n_iter - 1) & 1);
          ptx::tc_fence_after();
          const float f = grow ? ptx::ex2((m - m_new) * p.scale_log2) : 1.f;
          if (grow) { m = m_new; l *= f; }
#pragma unroll
          for (int ch = 0; ch < D / 32; ++ch) {
            uint32_t o[32];
            ptx::tmem_ld32(tO + ch * 32, o);
            ptx::tc_wait_ld();
#pragma unroll
            for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * f);
            ptx::tmem_st32(tO + ch * 32, o);
          }
        }
        const float neg_ms = (m == -INFINITY) ? 0.f : -m * p.scale_log2;
        // P = 2^(s*scale - m*scale) in kPChunks chunks; each chunk is handed to the MMA warp as soon
        // as it sits in TMEM, so that P.V of the early chunks overlaps the exponentials of the later ones.
        // Tiles in which some row of this warp has masked keys take the all-MUFU variant: ex2(-inf) is
        // exactly 0 there, while the polynomial clamps to 2^-126 (an empty row must sum to l == 0, R11).
        const float2 sc2 = make_float2(p.scale_log2, p.scale_log2), nm2 = make_float2(neg_ms, neg_ms);
        float2 sumA = make_float2(0.f, 0.f), sumB = make_float2(0.f, 0.f);
        auto exp_halves = [&](auto poly_tag) {
          constexpr unsigned kPoly = decltype(poly_tag)::value;
#pragma unroll
          for (int u = 0; u < kBlockN / 16; ++u) {  // 16 keys -> 8 packed BF16 pairs -> 8 TMEM columns
            uint32_t pk[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const int key = u * 16 + 2 * i;
              const float2 x = ptx::fma2(make_float2(__uint_as_float(s[key >> 5][key & 31]), __uint_as_float(s[key >> 5][(key & 31) + 1])), sc2, nm2);
              float2 e;
              if ((kPoly >> ((u & 1) * 8 + i)) & 1u) e = ptx::ex2_poly2(x);
              else e = make_float2(ptx::ex2(x.x), ptx::ex2(x.y));
              if (i & 1) sumB = ptx::add2(sumB, e); else sumA = ptx::add2(sumA, e);
              pk[i] = ptx::pack_bf16(e.x, e.y);
            }
            ptx::tmem_st8(tS + u * 8, pk);
            if (chunk_ending_at(u + 1) >= 0) {  // compile-time: the loop is fully unrolled
              ptx::tc_wait_st();
              ptx::tc_fence_before();
              ptx::mbar_arrive(p_ready + chunk_ending_at(u + 1) * 8);
            }
          }
        };
        if (__any_sync(0xffffffffu, lim < kBlockN)) exp_halves(std::integral_constant<unsigned, 0u>{});
        else exp_halves(std::integral_constant<unsigned, kPolyMask>{});
        const float2 sum2 = ptx::add2(sumA, sumB);
        l += sum2.x + sum2.y;
      }

      // ------------------------------ segment epilogue ------------------------------
      ptx::mbar_wait(o_done, (n_iter - 1) & 1);
      ptx::tc_fence_after();
      const float m_l2 = m == -INFINITY ? -INFINITY : m * p.scale_log2;  // running max in log2 units
      if (sp.whole && !sp.single) {
        const float inv = l > 0.f ? 1.f / l : 0.f;
        if (p.lse != nullptr && row_valid) p.lse[(int64_t)g.head * p.Lq + row] = l > 0.f ? (ptx::lg2(l) + m_l2) * kLn2 : -INFINITY;
        store_row(g.head, row, inv, tO, [](int, uint32_t (&)[32]) {});
      } else if (sp.whole) {
        // single unit, whole KV range in this CTA: slot 1 publishes (m, l) and keeps its accumulator in TMEM; slot 0's
        // thread of the same row (same TMEM lane) merges the two halves and writes the final row.
        if (tile == 1) {
          merge_ml[row_in_tile] = make_float2(m_l2, l);
          ptx::tc_fence_before();
          ptx::named_bar_arrive(1, 2 * kBlockM);  // "slot 1's half is complete"
          ptx::named_bar_sync(2, 2 * kBlockM);    // slot 0 has read O1: the next segment may overwrite it
        } else {
          ptx::named_bar_sync(1, 2 * kBlockM);
          ptx::tc_fence_after();
          const float2 other = merge_ml[row_in_tile];
          const float M = fmaxf(m_l2, other.x);
          const float w0 = M == -INFINITY ? 0.f : ptx::ex2(m_l2 - M), w1 = M == -INFINITY ? 0.f : ptx::ex2(other.x - M);
          const float L = w0 * l + w1 * other.y;
          const float inv = L > 0.f ? 1.f / L : 0.f;
          if (p.lse != nullptr && row_valid) p.lse[(int64_t)g.head * p.Lq + row] = L > 0.f ? (ptx::lg2(L) + M) * kLn2 : -INFINITY;
          const uint32_t tO1 = tmem + C::kTmemO1 + lane_off;
          store_row(g.head, row, inv, tO, [&](int ch, uint32_t (&o)[32]) {
            uint32_t o1[32];
            ptx::tmem_ld32(tO1 + ch * 32, o1);
            ptx::tc_wait_ld();
#pragma unroll
            for (int c = 0; c < 32; ++c) {
              // a half that saw no key (w == 0) may hold an accumulator that was never written: keep it out
              const float a0 = w0 > 0.f ? w0 * __uint_as_float(o[c]) : 0.f, a1 = w1 > 0.f ? w1 * __uint_as_float(o1[c]) : 0.f;
              o[c] = __float_as_uint(a0 + a1);
            }
          });
          ptx::tc_fence_before();
          ptx::named_bar_arrive(2, 2 * kBlockM);
        }
      } else {
        // partial: unnormalised O (FP32), running max (log2 units) and sum, into record (item + cta) * 2 + slot
        const int64_t rec = ((int64_t)g.head * p.n_units + g.unit + blockIdx.x) * 2 + tile;
        if (row_valid) p.part_ml[rec * kBlockM + row_in_tile] = make_float2(m_l2, l);
        float4* po = reinterpret_cast<float4*>(p.part_o) + rec * (D / 4) * kBlockM + row_in_tile;
#pragma unroll
        for (int ch = 0; ch < D / 32; ++ch) {
          uint32_t o[32];
          ptx::tmem_ld32(tO + ch * 32, o);
          ptx::tc_wait_ld();
          if (row_valid) {  // padding rows are never read by the combine kernel
#pragma unroll
            for (int c = 0; c < 8; ++c)
              po[(int64_t)(ch * 8 + c) * kBlockM] = make_float4(__uint_as_float(o[4 * c]), __uint_as_float(o[4 * c + 1]),
                                                                __uint_as_float(o[4 * c + 2]), __uint_as_float(o[4 * c + 3]));
          }
        }
      }
      // the next segment's first P.V overwrites O: order our TMEM reads before the p_ready arrive that unleashes it
      ptx::tc_fence_before();
    }
  }

  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) ptx::tmem_dealloc(tmem, kTmemCols);
}

// ---------------------------------------------------------------------------------------------
// combine kernel: merges the split-KV partials of the phase-2 units, and zero-fills phase-2 units
// that see no key at all.  grid = (number of phase-2 units, d/4), block = 256 threads: thread r handles
// row r % 128 of tile slot r / 128 (a single unit has one Q tile: its slot-1 threads have nothing to do).
// ---------------------------------------------------------------------------------------------
template <int D, bool OUT_F32, int kBatch>
__global__ void __launch_bounds__(kPairM) attn_combine_kernel(const __grid_constant__ Params p) {
  wsi::pdl_trigger();
  wsi::pdl_wait();  // the partials are the attention kernel's
  const int w = p.n_waves * p.grid + blockIdx.x, head = w / p.n_units, unit = w - head * p.n_units;
  const int q4 = blockIdx.y, slot = threadIdx.x >> 7, r = threadIdx.x & (kBlockM - 1);
  const bool single = p.last_single && unit == p.n_units - 1;
  if (single && slot == 1) return;
  const int row = (2 * unit + slot) * kBlockM + r;
  if (row >= p.Lq) return;
  const int Tp = p.unit_prefix[p.n_units];
  const int n_iters = p.unit_prefix[unit + 1] - p.unit_prefix[unit];
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  float lse = -INFINITY;
  if (n_iters > 0) {
    const int64_t a = (int64_t)head * Tp + p.unit_prefix[unit];
    const int c_lo = cta_of_iter(p, a), c_hi = cta_of_iter(p, a + n_iters - 1);
    if (c_lo == c_hi) return;  // one CTA covered the whole KV range and wrote the final rows itself
    // records (w + c) * 2 + s: a pair's tile slot s has one record per CTA (stride 2); a single unit's tile has both
    // slots' records of every CTA (stride 1)
    const int64_t rec0 = ((int64_t)w + c_lo) * 2 + (single ? 0 : slot);
    const int n_rec = (c_hi - c_lo + 1) * (single ? 2 : 1), stride = single ? 1 : 2;
    // online LSE-weighted merge, kBatch partials per step with all 2 kBatch loads of a step in flight at once (the kernel is a
    // chain of dependent L2 round trips otherwise).  Four per step when every item has few partials (cfg2, cfg4: eight cost
    // occupancy and measured slower there), eight when some item has more than eight (cfg3, cfg5: 12-13 partials per item).
    float M = -INFINITY, L = 0.f;
    for (int k = 0; k < n_rec; k += kBatch) {
      float2 ml[kBatch];
      float4 o[kBatch];
#pragma unroll
      for (int u = 0; u < kBatch; ++u) {
        ml[u] = make_float2(-INFINITY, 0.f);
        o[u] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (k + u < n_rec && !pool_empty(p, c_lo + (single ? (k + u) >> 1 : k + u))) {  // an empty CTA inside the span wrote no record
          const int64_t rec = rec0 + (int64_t)(k + u) * stride;
          ml[u] = p.part_ml[rec * kBlockM + r];
          o[u] = reinterpret_cast<const float4*>(p.part_o)[(rec * (D / 4) + q4) * kBlockM + r];
        }
      }
      float M_new = M;
#pragma unroll
      for (int u = 0; u < kBatch; ++u) M_new = fmaxf(M_new, ml[u].x);
      if (M_new > -INFINITY) {
        const float f = ptx::ex2(M - M_new);  // 0 while nothing has been merged yet (M = -inf)
        acc.x *= f; acc.y *= f; acc.z *= f; acc.w *= f;
        L *= f;
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
          if (ml[u].x == -INFINITY) continue;  // a partial that saw no key: weight 0, accumulator not meaningful
          const float wgt = ptx::ex2(ml[u].x - M_new);
          acc.x += wgt * o[u].x; acc.y += wgt * o[u].y; acc.z += wgt * o[u].z; acc.w += wgt * o[u].w;
          L += wgt * ml[u].y;
        }
        M = M_new;
      }
    }
    if (L > 0.f) {
      const float inv = 1.f / L;
      acc.x *= inv; acc.y *= inv; acc.z *= inv; acc.w *= inv;
      lse = (ptx::lg2(L) + M) * kLn2;
    } else {
      acc = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  }
  const RowDst rd = row_dst(p, row);
  const int64_t o_off = rd.elem_off + (int64_t)head * D + q4 * 4;
  for (int k = 0; k < rd.n_dst; ++k) {
    if constexpr (OUT_F32) {
      *reinterpret_cast<float4*>(reinterpret_cast<float*>(p.out_peer[rd.peer0 + k]) + o_off) = acc;
    } else {
      uint2 v;
      v.x = ptx::pack_bf16(acc.x, acc.y);
      v.y = ptx::pack_bf16(acc.z, acc.w);
      *reinterpret_cast<uint2*>(reinterpret_cast<__nv_bfloat16*>(p.out_peer[rd.peer0 + k]) + o_off) = v;
    }
  }
  if (q4 == 0 && p.lse != nullptr) p.lse[(int64_t)head * p.Lq + row] = lse;
}

// FP32 -> BF16 staging for WS_DTYPE_F32 inputs (config 1; R9).
// Copies n_planes planes of plane_elems contiguous floats; planes are src_plane_pitch floats / dst_plane_pitch BF16 elements apart.
__global__ void cast_f32_to_bf16_kernel(__nv_bfloat16* __restrict__ dst, const float* __restrict__ src, int64_t n_planes,
                                        int64_t plane_elems, int64_t src_plane_pitch, int64_t dst_plane_pitch) {
  wsi::pdl_trigger();
  wsi::pdl_wait();
  const int64_t total = n_planes * plane_elems;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t pl = i / plane_elems, e = i - pl * plane_elems;
    dst[pl * dst_plane_pitch + e] = __float2bfloat16_rn(src[pl * src_plane_pitch + e]);
  }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
PFN_cuTensorMapEncodeTiled_v12000 get_encode_fn() {
  static PFN_cuTensorMapEncodeTiled_v12000 fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(f);
  });
  return fn;
}

// 3-D BF16 tensor map, 128-byte swizzle, box = {64 elements, b1, b2}.
bool encode_map(CUtensorMap* map, const void* base, uint64_t d0, uint64_t d1, uint64_t d2, uint64_t stride1_bytes,
                uint64_t stride2_bytes, uint32_t b1, uint32_t b2) {
  auto fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[3] = {d0, d1, d2};
  cuuint64_t strides[2] = {stride1_bytes, stride2_bytes};
  cuuint32_t box[3] = {64, b1, b2};
  cuuint32_t estr[3] = {1, 1, 1};
  return fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// 3-D UINT8 tensor map of an FP8 cache [H, capacity, d] (valid rows [0, cache_len)), no swizzle, box = {d bytes, 128 rows, 1}.
bool encode_map_u8(CUtensorMap* map, const void* base, uint64_t d, uint64_t rows, uint64_t H, uint64_t capacity) {
  auto fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[3] = {d, rows, H};
  cuuint64_t strides[2] = {d, d * capacity};
  cuuint32_t box[3] = {(cuuint32_t)d, kBlockN, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  return fn(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Per-device state: the SM count and which kernel instantiations already carry their dynamic shared-memory
// attribute on that device (cudaFuncSetAttribute is per device).  Indexed by cudaGetDevice(), like ws_unit.cu's pipes.
constexpr int kMaxDevices = 64;
constexpr int kKernelVariants = 8;
struct DeviceState {
  int sms = 0;
  bool attr_set[kKernelVariants] = {};
};
std::mutex g_dev_mu;
DeviceState g_dev[kMaxDevices];

// The current device's slot with its SM count filled in, or nullptr (no device / index beyond the table).
DeviceState* device_state(cudaError_t* err) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess && (dev < 0 || dev >= kMaxDevices)) e = cudaErrorInvalidDevice;
  if (e == cudaSuccess) {
    std::lock_guard<std::mutex> lock(g_dev_mu);
    DeviceState& st = g_dev[dev];
    if (st.sms == 0) {
      int v = 0;
      e = cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
      if (e == cudaSuccess && v <= 0) e = cudaErrorNoDevice;
      if (e == cudaSuccess) st.sms = v;
    }
    if (e == cudaSuccess) return &st;
  }
  if (err) *err = e;
  return nullptr;
}

// Sets MaxDynamicSharedMemorySize on `kernel` once per device.
template <typename K>
cudaError_t ensure_smem_attr(DeviceState* st, int variant, K kernel, int bytes) {
  std::lock_guard<std::mutex> lock(g_dev_mu);
  if (st->attr_set[variant]) return cudaSuccess;
  const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e == cudaSuccess) st->attr_set[variant] = true;
  return e;
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct WsLayout {
  size_t part_o, part_ml, stage_q, stage_kc, stage_vc, stage_kn, stage_vn, total;
};

WsLayout ws_layout(int32_t Lq, int32_t H, int32_t d, int64_t kv_total, int64_t cache_len, int32_t Ln, ws_dtype dt,
                   bool exact) {
  WsLayout L{};
  const size_t n_units = (size_t)(Lq + kPairM - 1) / kPairM;
  const size_t slots = n_units * H + kMaxCtas;  // x 2 records of 128 rows each
  size_t off = 0;
  L.part_o = off; off = align_up(off + slots * kPairM * (size_t)d * 4, 256);
  L.part_ml = off; off = align_up(off + slots * kPairM * 8, 256);
  if (dt == WS_DTYPE_F32) {
    L.stage_q = off; off = align_up(off + (size_t)Lq * H * d * 2, 256);
    if (exact) {
      L.stage_kc = off; off = align_up(off + (size_t)H * cache_len * d * 2, 256);
      L.stage_vc = off; off = align_up(off + (size_t)H * cache_len * d * 2, 256);
      L.stage_kn = off; off = align_up(off + (size_t)Ln * H * d * 2, 256);
      L.stage_vn = off; off = align_up(off + (size_t)Ln * H * d * 2, 256);
    } else {  // size query: only cache_len + Ln is known; each of the four regions may need its own rounding
      off = align_up(off + 2 * (size_t)H * kv_total * d * 2, 256) + 4 * 256;
    }
  }
  L.total = off;
  return L;
}

#ifndef WS_COMBINE_BATCH8_FROM
#define WS_COMBINE_BATCH8_FROM 9
#endif
template <int D, bool OUT_F32, bool KV8>
int launch_attention(const Params& prm, DeviceState* st, cudaStream_t stream) {
  using C = Cfg<D, KV8>;
  const cudaError_t ae = ensure_smem_attr(st, (D == 128 ? 0 : 3) + (KV8 ? 2 : (OUT_F32 ? 1 : 0)), attn_fwd_kernel<D, OUT_F32, KV8>, C::kSmemBytes);
  if (ae != cudaSuccess) return wsi::cuda_fail(ae);
  int launches = 0;
  if (prm.grid > 0) {
    const cudaError_t e = wsi::launch_pdl(attn_fwd_kernel<D, OUT_F32, KV8>, dim3(prm.grid), dim3(C::kThreadsCta), C::kSmemBytes, stream, prm);
    if (e != cudaSuccess) return wsi::cuda_fail(e);
    ++launches;
  }
  const int n_pool_items = prm.H * prm.n_units - prm.n_waves * prm.grid;
  if (n_pool_items > 0 && prm.combine_items > 0) {
    dim3 cgrid((unsigned)n_pool_items, D / 4);  // items on x: H * n_units may exceed the 65535 limit of y
    const cudaError_t e = prm.combine_max_rec >= WS_COMBINE_BATCH8_FROM ? wsi::launch_pdl(attn_combine_kernel<D, OUT_F32, 8>, cgrid, dim3(kPairM), 0, stream, prm)
                                                  : wsi::launch_pdl(attn_combine_kernel<D, OUT_F32, 4>, cgrid, dim3(kPairM), 0, stream, prm);
    if (e != cudaSuccess) return wsi::cuda_fail(e);
    ++launches;
  }
  return wsi::after_launch(launches);
}

}  // namespace

extern "C" __attribute__((visibility("default"))) size_t ws_block_causal_attn_workspace_bytes(int32_t Lq, int32_t H, int32_t d, int64_t kv_total, ws_dtype dt) {
  if (Lq <= 0 || H <= 0 || d <= 0 || kv_total < 0) return 0;
  return ws_layout(Lq, H, d, kv_total, 0, 0, dt, false).total;
}

namespace {
// The cache part of the key timeline as physical runs of the cache tensor (a ring's window wraps at most once): run A =
// rows [ring_start, ring_start + len_a), run B = rows [0, cache_len - len_a).  Each run is tiled on its own (its last tile
// may be partial), so the timeline has n_tiles_a + n_tiles_b cache tiles.  A linear cache is the case ring_start = 0.
struct CacheRuns {
  int64_t len_a, len_b;
  int n_tiles_a, n_tiles_b;
};
CacheRuns cache_runs(int64_t capacity, int64_t ring_start, int64_t cache_len) {
  CacheRuns r;
  r.len_a = ring_start + cache_len <= capacity || ring_start == 0 ? cache_len : capacity - ring_start;
  r.len_b = cache_len - r.len_a;
  r.n_tiles_a = (int)((r.len_a + kBlockN - 1) / kBlockN);
  r.n_tiles_b = (int)((r.len_b + kBlockN - 1) / kBlockN);
  return r;
}

// KV tiles the last row of Q tile `qt` can see (a tile visits exactly those).
int64_t kv_tiles_of_q_tile(const ws_block_mask* mask, int32_t Lq, int64_t cache_len, const CacheRuns& runs, int qt) {
  const int last_row = ((qt + 1) * kBlockM < Lq ? (qt + 1) * kBlockM : Lq) - 1;
  int b = 0;
  while (last_row >= mask->q_block_end[b]) ++b;
  const int64_t nvis = mask->kv_visible[b];
  if (nvis <= 0) return 0;
  if (nvis <= runs.len_a) return (nvis + kBlockN - 1) / kBlockN;
  if (nvis <= cache_len) return runs.n_tiles_a + (nvis - runs.len_a + kBlockN - 1) / kBlockN;
  return runs.n_tiles_a + runs.n_tiles_b + (nvis - cache_len + kBlockN - 1) / kBlockN;
}

// Work units of a head and their iteration counts: Q tiles (2u, 2u + 1) form pair unit u, which runs one iteration
// per KV tile its later tile sees; an odd last Q tile is a single unit, whose KV tiles are cut in two runs (one per
// tile slot), i.e. one iteration per two KV tiles.  Fills prm.unit_prefix / n_cache_tiles / last_* (needs
// prm.n_units) and returns the iterations per head.  unit_kv_tiles (optional): KV tiles each unit visits.
int64_t build_unit_prefix(Params& prm, const ws_block_mask* mask, int32_t Lq, int64_t cache_len, int32_t* unit_kv_tiles) {
  const CacheRuns runs = cache_runs(prm.capacity, prm.ring_start, cache_len);
  prm.len_a = runs.len_a;
  prm.n_tiles_a = runs.n_tiles_a;
  prm.n_cache_tiles = runs.n_tiles_a + runs.n_tiles_b;
  const int n_q_tiles = (Lq + kBlockM - 1) / kBlockM;
  prm.last_single = n_q_tiles & 1;
  prm.last_kv_tiles = 0;
  int64_t Tp = 0;
  prm.unit_prefix[0] = 0;
  for (int u = 0; u < prm.n_units; ++u) {
    const bool single = prm.last_single && u == prm.n_units - 1;
    const int64_t n = kv_tiles_of_q_tile(mask, Lq, cache_len, runs, single ? 2 * u : 2 * u + 1);
    if (single) prm.last_kv_tiles = (int32_t)n;
    if (unit_kv_tiles) unit_kv_tiles[u] = (int32_t)n;
    Tp += single ? (n + 1) / 2 : n;
    prm.unit_prefix[u + 1] = (int32_t)Tp;
  }
  return Tp;
}

// Cost model of the schedule, in hundredths of an iteration (measured on B200 with a device-side clock trace,
// profiles/r02_attn_ncu.md): every segment a CTA starts costs about two iterations (Q load and the first Q.K^T
// before any softmax can run, accumulator read-out at the end).  An iteration of a single unit moves two separate K/V
// tiles instead of one shared one; its extra cost was within the noise of the fit (cfg4: 1.58 vs 1.57 us), so both
// kinds of iteration count the same.
constexpr int64_t kCostPairIter = 100, kCostSingleIter = 100, kCostSegment = 200;

// Contiguous partition of the flattened iterations [t_begin, T) over the CTAs such that no CTA's cost (its phase-1
// cost p1cost[c] plus segment and iteration costs of its share) exceeds `budget`.  Fills begin[0..G] and returns
// whether everything fitted.
bool partition_pool(const Params& prm, int64_t Tp, int64_t t_begin, int64_t T, int64_t G, const int64_t* p1cost, int64_t budget,
                    int64_t* begin) {
  const int n_units = prm.n_units;
  int64_t t = t_begin;
  for (int64_t c = 0; c < G; ++c) {
    begin[c] = t;
    int64_t left = budget - p1cost[c];
    while (t < T) {
      const int64_t rem = t % Tp;
      int u = 0;
      while (u + 1 < n_units && prm.unit_prefix[u + 1] <= rem) ++u;  // unit holding rem (empty units have no iterations)
      while (prm.unit_prefix[u + 1] == prm.unit_prefix[u]) ++u;
      const int64_t per_iter = (prm.last_single && u == n_units - 1) ? kCostSingleIter : kCostPairIter;
      const int64_t in_unit = prm.unit_prefix[u + 1] - rem;
      if (left < kCostSegment + per_iter) break;
      left -= kCostSegment;
      const int64_t n = left / per_iter < in_unit ? left / per_iter : in_unit;
      t += n;
      left -= n * per_iter;
      if (n < in_unit) break;
    }
  }
  begin[G] = t;
  return t == T;
}

// Pool items the combine kernel has work for: those that see no key (zero fill) and those split over several CTAs.
// Fills prm.combine_items (0: the combine kernel is not launched).
void count_combine_items(Params& prm) {
  const int n_units = prm.n_units;
  const int64_t n_items = (int64_t)prm.H * n_units, Tp = prm.unit_prefix[n_units];
  const int G = prm.grid;
  auto cta_of = [&](int64_t t) {
    int lo = 0, hi = G - 1;
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (prm.pool_begin[mid] <= t) lo = mid; else hi = mid - 1;
    }
    return lo;
  };
  int32_t n = 0, max_rec = 0;
  for (int64_t w = (int64_t)prm.n_waves * G; w < n_items; ++w) {
    const int u = (int)(w % n_units);
    const int64_t iters = prm.unit_prefix[u + 1] - prm.unit_prefix[u];
    if (iters == 0) { ++n; continue; }
    const int64_t a = (w / n_units) * Tp + prm.unit_prefix[u];
    const int span = cta_of(a + iters - 1) - cta_of(a) + 1;
    if (span > 1) {
      ++n;
      const int rec = span * ((prm.last_single && u == n_units - 1) ? 2 : 1);
      max_rec = rec > max_rec ? rec : max_rec;
    }
  }
  prm.combine_items = n;
  prm.combine_max_rec = max_rec;
}

// The two-phase schedule (see Params) for a device with `sms` SMs: fills prm.grid, n_waves, pool_begin, combine_items.
void build_schedule(Params& prm, int64_t Tp, int sms) {
  const int n_units = prm.n_units, H = prm.H;
  const int64_t T = Tp * H, n_items = (int64_t)H * n_units;
  int64_t G = T > 0 ? T : n_items;
  if (G > sms) G = sms;
  if (G > kMaxCtas) G = kMaxCtas;
  prm.grid = (int32_t)G;
  if (T == 0) {  // nothing visible anywhere: every item is a (zero-filling) phase-1 item
    prm.n_waves = (int32_t)((n_items + G - 1) / G);
    for (int64_t c = 0; c <= G; ++c) prm.pool_begin[c] = 0;
    prm.combine_items = 0;
    prm.combine_max_rec = 0;
    return;
  }
  auto item_cost = [&](int64_t i) {
    const int u = (int)(i % n_units);
    const int64_t n = prm.unit_prefix[u + 1] - prm.unit_prefix[u];
    return n == 0 ? (int64_t)0 : kCostSegment + n * ((prm.last_single && u == n_units - 1) ? kCostSingleIter : kCostPairIter);
  };
  auto item_flat = [&](int64_t i) { return (i / n_units) * Tp + prm.unit_prefix[i % n_units]; };
  // smallest per-CTA budget for which the pool [t_begin, T) fits next to the phase-1 costs
  auto min_budget = [&](int64_t t_begin, const int64_t* p1cost, int64_t* begin) {
    int64_t lo = 0, hi = 0;
    for (int64_t c = 0; c < G; ++c) lo = p1cost[c] > lo ? p1cost[c] : lo;
    hi = lo + (T - t_begin) * kCostSingleIter + kCostSegment * (n_items + 1) + 1;
    while (lo < hi) {
      const int64_t mid = (lo + hi) / 2;
      if (partition_pool(prm, Tp, t_begin, T, G, p1cost, mid, begin)) hi = mid; else lo = mid + 1;
    }
    partition_pool(prm, Tp, t_begin, T, G, p1cost, lo, begin);
    return lo;
  };
  int64_t zero[kMaxCtas] = {}, p1cost[kMaxCtas] = {}, begin_a[kMaxCtas + 1], begin_b[kMaxCtas + 1];
  // candidate A: pure stream-K over all items.  The even split in iterations is kept unless the cost-aware partition
  // (which shortens the share of CTAs that start more segments or run single-unit iterations) models > 5 % faster:
  // with long segments the even split was measured marginally better (cfg4), with short ones clearly worse (cfg2).
  int64_t makespan_a = min_budget(0, zero, begin_a);
  {
    int64_t even[kMaxCtas + 1], worst = 0;
    for (int64_t c = 0; c <= G; ++c) even[c] = (c * T) / G;
    for (int64_t c = 0; c < G; ++c) {
      int64_t cost = 0;
      for (int64_t t = even[c]; t < even[c + 1];) {
        const int64_t rem = t % Tp;
        int u = 0;
        while (u + 1 < n_units && prm.unit_prefix[u + 1] <= rem) ++u;
        while (prm.unit_prefix[u + 1] == prm.unit_prefix[u]) ++u;
        const int64_t in_unit = prm.unit_prefix[u + 1] - rem, n = in_unit < even[c + 1] - t ? in_unit : even[c + 1] - t;
        cost += kCostSegment + n * ((prm.last_single && u == n_units - 1) ? kCostSingleIter : kCostPairIter);
        t += n;
      }
      worst = cost > worst ? cost : worst;
    }
    if (makespan_a * 105 >= worst * 100) {
      makespan_a = worst;
      for (int64_t c = 0; c <= G; ++c) begin_a[c] = even[c];
    }
  }
  // candidate B: W whole-item waves, the remaining items pooled
  const int64_t W = n_items / G;
  bool use_b = false;
  if (W > 0) {
    for (int64_t c = 0; c < G; ++c)
      for (int64_t w = 0; w < W; ++w) p1cost[c] += item_cost(w * G + c);
    const int64_t makespan_b = min_budget(item_flat(W * G), p1cost, begin_b);
    // B trades a slightly longer critical path for far fewer split items and L2 reuse of K/V across the units of a head
    // (measured on B200, cfg4: modelled 4-5 % longer, 3.5 % FASTER -- 265.0 us against 274.5 for pure stream-K, whose every item
    // writes partials for the combine kernel; the slack was 3 % until then.  cfg2 / cfg3 / cfg5 do not depend on it.)
    use_b = makespan_b * 100 <= makespan_a * 106;
  }
  prm.n_waves = use_b ? (int32_t)W : 0;
  for (int64_t c = 0; c <= G; ++c) prm.pool_begin[c] = use_b ? begin_b[c] : begin_a[c];
  count_combine_items(prm);
}

// The schedule depends on the problem shape only (Lq, H, cache_len, Ln, mask, SM count): a streaming session repeats
// the same shape for every layer and denoising step, so the last few schedules are kept (per host thread).
struct ScheduleKey {
  int32_t Lq, H, Ln, n_blocks, sms;
  int64_t cache_len, capacity, ring_start;
  int32_t q_block_end[WS_MAX_MASK_BLOCKS], kv_visible[WS_MAX_MASK_BLOCKS];
};
struct ScheduleEntry {
  bool valid = false;
  uint64_t stamp = 0;
  ScheduleKey key;
  int32_t n_cache_tiles, n_tiles_a, last_single, last_kv_tiles, n_waves, grid, combine_items, combine_max_rec;
  int64_t len_a;
  int32_t unit_prefix[kMaxUnits + 1];
  int64_t pool_begin[kMaxCtas + 1];
};
// Fills the schedule fields of prm (needs Lq, H, Ln, cache_len, n_units set); returns the iterations per head.
int64_t schedule_for(Params& prm, const ws_block_mask* mask, int sms) {
  constexpr int kEntries = 8;
  thread_local ScheduleEntry cache[kEntries];
  thread_local uint64_t clock = 0;
  ScheduleKey key;
  memset(&key, 0, sizeof(key));
  key.Lq = prm.Lq; key.H = prm.H; key.Ln = prm.Ln; key.n_blocks = mask->n_blocks; key.sms = sms; key.cache_len = prm.cache_len;
  key.ring_start = prm.ring_start; key.capacity = prm.ring_start ? prm.capacity : 0;  // a linear cache's schedule does not depend on its capacity
  for (int b = 0; b < mask->n_blocks; ++b) { key.q_block_end[b] = mask->q_block_end[b]; key.kv_visible[b] = mask->kv_visible[b]; }
  ScheduleEntry* victim = &cache[0];
  for (ScheduleEntry& e : cache) {
    if (e.valid && memcmp(&e.key, &key, sizeof(key)) == 0) {
      e.stamp = ++clock;
      prm.n_cache_tiles = e.n_cache_tiles; prm.n_tiles_a = e.n_tiles_a; prm.len_a = e.len_a;
      prm.last_single = e.last_single; prm.last_kv_tiles = e.last_kv_tiles;
      prm.n_waves = e.n_waves; prm.grid = e.grid; prm.combine_items = e.combine_items; prm.combine_max_rec = e.combine_max_rec;
      memcpy(prm.unit_prefix, e.unit_prefix, sizeof(int32_t) * (prm.n_units + 1));
      memcpy(prm.pool_begin, e.pool_begin, sizeof(int64_t) * (e.grid + 1));
      return prm.unit_prefix[prm.n_units];
    }
    if (!e.valid || e.stamp < victim->stamp || (victim->valid && !e.valid)) victim = &e;
  }
  const int64_t Tp = build_unit_prefix(prm, mask, prm.Lq, prm.cache_len, nullptr);
  build_schedule(prm, Tp, sms);
  victim->valid = true; victim->stamp = ++clock; victim->key = key;
  victim->n_cache_tiles = prm.n_cache_tiles; victim->n_tiles_a = prm.n_tiles_a; victim->len_a = prm.len_a;
  victim->last_single = prm.last_single; victim->last_kv_tiles = prm.last_kv_tiles;
  victim->n_waves = prm.n_waves; victim->grid = prm.grid; victim->combine_items = prm.combine_items; victim->combine_max_rec = prm.combine_max_rec;
  memcpy(victim->unit_prefix, prm.unit_prefix, sizeof(int32_t) * (prm.n_units + 1));
  memcpy(victim->pool_begin, prm.pool_begin, sizeof(int64_t) * (prm.grid + 1));
  return Tp;
}

// The mask rules shared by the attention entry points and the schedule diagnostic.
int check_mask(const ws_block_mask* mask, int32_t Lq, int64_t cache_len, int32_t Ln) {
  if (!mask || mask->n_blocks <= 0 || !mask->q_block_end || !mask->kv_visible) return WS_ERR_INVALID_ARG;
  if (mask->n_blocks > WS_MAX_MASK_BLOCKS) return WS_ERR_UNSUPPORTED;
  int32_t prev_end = 0, prev_vis = 0;
  for (int b = 0; b < mask->n_blocks; ++b) {
    if (mask->q_block_end[b] <= prev_end || mask->kv_visible[b] < prev_vis) return WS_ERR_INVALID_ARG;
    if ((int64_t)mask->kv_visible[b] > cache_len + Ln) return WS_ERR_OUT_OF_RANGE;
    prev_end = mask->q_block_end[b];
    prev_vis = mask->kv_visible[b];
  }
  return prev_end == Lq ? WS_OK : WS_ERR_INVALID_ARG;
}
}  // namespace

// Host-only diagnostic: the schedule ws_block_causal_attn uses for this problem on a device with n_sms SMs.
extern "C" __attribute__((visibility("default"))) int ws_attn_schedule(int32_t Lq, int32_t H, int64_t cache_len, int32_t Ln, const ws_block_mask* mask,
                                int32_t n_sms, int32_t* grid, int32_t* n_waves, int32_t* unit_iters, int32_t* unit_kv_tiles,
                                int64_t* pool_begin) {
  if (Lq <= 0 || H <= 0 || cache_len < 0 || Ln < 0 || n_sms <= 0 || !grid || !n_waves || !unit_iters || !unit_kv_tiles || !pool_begin)
    return WS_ERR_INVALID_ARG;
  if (const int rc = check_mask(mask, Lq, cache_len, Ln)) return rc;
  if (cache_len + Ln > 0x7fffffffLL / kMaxUnits - kBlockN) return WS_ERR_UNSUPPORTED;
  Params* prm = new Params();
  prm->Lq = Lq; prm->H = H; prm->Ln = Ln; prm->cache_len = cache_len;
  prm->n_units = (Lq + kPairM - 1) / kPairM;
  if (prm->n_units > kMaxUnits) { delete prm; return WS_ERR_UNSUPPORTED; }
  const int64_t Tp = build_unit_prefix(*prm, mask, Lq, cache_len, unit_kv_tiles);
  build_schedule(*prm, Tp, n_sms);
  *grid = prm->grid;
  *n_waves = prm->n_waves;
  for (int u = 0; u < prm->n_units; ++u) unit_iters[u] = prm->unit_prefix[u + 1] - prm->unit_prefix[u];
  for (int c = 0; c <= prm->grid; ++c) pool_begin[c] = prm->pool_begin[c];
  delete prm;
  return WS_OK;
}

// Every argument check of the attention entry points.  Pure host logic: touches no device and launches nothing,
// so callers that enqueue other work first (ws_unit_forward_host) can run it up front.
int wsi::attn_validate(const void* out, const float* lse, const void* q, const void* k_cache, const void* v_cache, int64_t capacity,
                       int64_t cache_len, const void* k_new, const void* v_new, int32_t Ln, int32_t H, int32_t d, int32_t Lq,
                       const ws_block_mask* mask, float softmax_scale, const void* workspace, size_t workspace_bytes, ws_dtype dt) {
  if (dt != WS_DTYPE_BF16 && dt != WS_DTYPE_F32) return WS_ERR_UNSUPPORTED;
  if (d != 64 && d != 128) return WS_ERR_UNSUPPORTED;
  if (!out || !q || !mask || H <= 0 || Lq <= 0 || Ln < 0 || capacity < 0 || cache_len < 0) return WS_ERR_INVALID_ARG;
  if (!(softmax_scale >= 0.f) || !(softmax_scale < INFINITY)) return WS_ERR_INVALID_ARG;
  if ((Ln > 0) != (k_new != nullptr) || (Ln > 0) != (v_new != nullptr)) return WS_ERR_INVALID_ARG;
  if (cache_len > capacity) return WS_ERR_OUT_OF_RANGE;
  if (cache_len > 0 && (!k_cache || !v_cache)) return WS_ERR_INVALID_ARG;
  if (cache_len + Ln > 0x7fffffffLL / kMaxUnits - kBlockN) return WS_ERR_UNSUPPORTED;  // unit_prefix is int32
  if (const int rc = check_mask(mask, Lq, cache_len, Ln)) return rc;
  if ((Lq + kPairM - 1) / kPairM > kMaxUnits) return WS_ERR_UNSUPPORTED;
  if (!wsi::aligned16(out) || !wsi::aligned16(q) || !wsi::aligned16(k_cache) || !wsi::aligned16(v_cache) ||
      !wsi::aligned16(k_new) || !wsi::aligned16(v_new) || (lse && (reinterpret_cast<uintptr_t>(lse) & 3)))
    return WS_ERR_ALIGNMENT;
  const WsLayout L = ws_layout(Lq, H, d, cache_len + Ln, cache_len, Ln, dt, true);
  if (!workspace || workspace_bytes < L.total) return WS_ERR_WORKSPACE;
  if (!wsi::aligned256(workspace)) return WS_ERR_WORKSPACE;
  return WS_OK;
}

namespace {
// Shared implementation.  q / k_new / v_new / out are token-major with `tok_heads` heads per token in memory, of which
// the H heads starting at the given base pointers take part (tok_heads == H for the plain [L, H, d] call).
int attn_impl(void* out, float* lse, const void* q, const void* k_cache, const void* v_cache, int64_t capacity,
              int64_t cache_len, const void* k_new, const void* v_new, int32_t Ln, int32_t H, int32_t d, int32_t Lq,
              const ws_block_mask* mask, float softmax_scale, void* workspace, size_t workspace_bytes, ws_dtype dt,
              void* stream_, int64_t tok_heads, const int8_t* k_exp = nullptr, const int8_t* v_exp = nullptr, int64_t ring_start = 0,
              void* const* peer_outs = nullptr, int32_t n_peers = 1, int64_t peer_rows = 0, bool f32_out_only = false) {
  cudaStream_t stream = (cudaStream_t)stream_;
  const bool kv8 = k_exp != nullptr;  // the cache holds E4M3 codes with per-row exponents (ws_block_causal_attn_fp8kv)
  // ---- validation, descriptors and schedule first: nothing is launched on any error ----
  if (const int rc = wsi::attn_validate(out, lse, q, k_cache, v_cache, capacity, cache_len, k_new, v_new, Ln, H, d, Lq, mask,
                                        softmax_scale, workspace, workspace_bytes, dt))
    return rc;
  if (ring_start < 0 || (ring_start > 0 && ring_start >= capacity)) return WS_ERR_OUT_OF_RANGE;
  if (ring_start > 0x7fffffffLL - cache_len - kBlockN) return WS_ERR_UNSUPPORTED;  // TMA row coordinates are int32
  const int n_units = (Lq + kPairM - 1) / kPairM;
  const WsLayout L = ws_layout(Lq, H, d, cache_len + Ln, cache_len, Ln, dt, true);
  if (!get_encode_fn()) return wsi::cuda_fail(cudaErrorNotSupported);
  cudaError_t dev_err = cudaErrorNoDevice;
  DeviceState* dev = device_state(&dev_err);
  if (!dev) return wsi::cuda_fail(dev_err);

  char* ws = reinterpret_cast<char*>(workspace);
  const bool f32 = dt == WS_DTYPE_F32;
  // WS_DTYPE_F32 (reading R9): the kernel reads BF16 copies staged in the workspace; the cache copy is compacted to cache_len rows
  const void* q_b = f32 ? ws + L.stage_q : q;
  const void* kc_b = f32 ? ws + L.stage_kc : k_cache;
  const void* vc_b = f32 ? ws + L.stage_vc : v_cache;
  const void* kn_b = f32 ? ws + L.stage_kn : k_new;
  const void* vn_b = f32 ? ws + L.stage_vn : v_new;
  const int64_t cap_b = f32 ? cache_len : capacity;
  // a ring's window: the staged FP32 copy is linearised by the cast kernels, the BF16 cache is read in place as two runs
  const CacheRuns runs = cache_runs(capacity, ring_start, cache_len);
  const int64_t ring_b = f32 ? 0 : ring_start;
  const int64_t map_rows = ring_b + cache_len < cap_b ? ring_b + cache_len : cap_b;  // rows past the window's end read as zero

  Params prm;
  memset(&prm, 0, sizeof(prm));
  const uint64_t row_b = (uint64_t)d * 2;
  const uint64_t tok_b = row_b * (uint64_t)(f32 ? H : tok_heads);  // token pitch of the BF16 operands
  bool ok = encode_map(&prm.map_q, q_b, d, H, Lq, row_b, tok_b, 1, kBlockM);
  // a source with no rows still needs a well-formed (never dereferenced) descriptor
  ok = ok && (Ln > 0 ? encode_map(&prm.map_kn, kn_b, d, H, Ln, row_b, tok_b, 1, kBlockN)
                     : encode_map(&prm.map_kn, q_b, d, H, Lq, row_b, tok_b, 1, kBlockN));
  ok = ok && (Ln > 0 ? encode_map(&prm.map_vn, vn_b, d, H, Ln, row_b, tok_b, 1, kBlockN)
                     : encode_map(&prm.map_vn, q_b, d, H, Lq, row_b, tok_b, 1, kBlockN));
  if (kv8 && cache_len > 0) {
    ok = ok && encode_map_u8(&prm.map_kc, kc_b, d, cache_len, H, cap_b) && encode_map_u8(&prm.map_vc, vc_b, d, cache_len, H, cap_b);
  } else {
    ok = ok && (cache_len > 0 ? encode_map(&prm.map_kc, kc_b, d, map_rows, H, row_b, row_b * cap_b, kBlockN, 1)
                              : encode_map(&prm.map_kc, q_b, d, H, Lq, row_b, tok_b, 1, kBlockN));
    ok = ok && (cache_len > 0 ? encode_map(&prm.map_vc, vc_b, d, map_rows, H, row_b, row_b * cap_b, kBlockN, 1)
                              : encode_map(&prm.map_vc, q_b, d, H, Lq, row_b, tok_b, 1, kBlockN));
  }
  if (!ok) return wsi::cuda_fail(cudaErrorInvalidValue);
  if (peer_outs) {  // ws_block_causal_attn_push_out: `out` is peer 0's pointer (validated like a plain output)
    for (int r = 0; r < n_peers; ++r) prm.out_peer[r] = peer_outs[r];
    prm.n_peers = n_peers;
    prm.peer_rows = (int32_t)peer_rows;
  } else {
    prm.out_peer[0] = out;
    prm.n_peers = 1;
    prm.peer_rows = 0x7fffffff;
  }
  prm.out_pitch = (peer_outs ? (int64_t)n_peers * H : tok_heads) * d;  // a peer's output rows hold the heads of all ranks
  prm.lse = lse;
  prm.part_o = reinterpret_cast<float*>(ws + L.part_o);
  prm.part_ml = reinterpret_cast<float2*>(ws + L.part_ml);
  prm.cache_len = cache_len;
  prm.capacity = f32 ? cache_len : capacity;
  prm.ring_start = ring_b;
  prm.k_exp = k_exp;
  prm.v_exp = v_exp;
  prm.Lq = Lq; prm.H = H; prm.Ln = Ln; prm.n_blocks = mask->n_blocks; prm.n_units = n_units;
  prm.n_cache_tiles = (int)((cache_len + kBlockN - 1) / kBlockN);
  prm.scale = softmax_scale;
  // clamped away from 0 so that a masked (-inf) logit times the scale stays -inf (softmax_scale == 0 is legal)
  prm.scale_log2 = fmaxf(softmax_scale * kLog2e, 1e-30f);
  for (int b = 0; b < mask->n_blocks; ++b) {
    prm.q_block_end[b] = mask->q_block_end[b];
    prm.kv_visible[b] = mask->kv_visible[b];
  }
  schedule_for(prm, mask, dev->sms);

  // ---- launches ----
  if (f32) {
    int launches = 0;
    cudaError_t ce = cudaSuccess;
    auto cast = [&](const void* dstp, int64_t dst_pitch, const void* srcp, int64_t planes, int64_t plane_elems, int64_t pitch) {
      const int64_t total = planes * plane_elems;
      if (total == 0 || ce != cudaSuccess) return;
      const int blocks = (int)((total + 255) / 256 < 4096 ? (total + 255) / 256 : 4096);
      ce = wsi::launch_pdl(cast_f32_to_bf16_kernel, dim3(blocks), dim3(256), 0, stream,
                           reinterpret_cast<__nv_bfloat16*>(const_cast<void*>(dstp)), reinterpret_cast<const float*>(srcp), planes,
                           plane_elems, pitch, dst_pitch);
      if (ce == cudaSuccess) ++launches;
    };
    const int64_t hd = (int64_t)H * d;
    cast(q_b, hd, q, Lq, hd, tok_heads * d);  // token by token: the staged copy is compact [Lq, H, d]
    // the cache window in timeline order: run A (from ring_start), then run B (from physical row 0)
    const float* kc_f = reinterpret_cast<const float*>(k_cache);
    const float* vc_f = reinterpret_cast<const float*>(v_cache);
    __nv_bfloat16* kc_s = reinterpret_cast<__nv_bfloat16*>(const_cast<void*>(kc_b));
    __nv_bfloat16* vc_s = reinterpret_cast<__nv_bfloat16*>(const_cast<void*>(vc_b));
    cast(kc_s, cache_len * d, kc_f + ring_start * d, H, runs.len_a * d, capacity * d);
    cast(vc_s, cache_len * d, vc_f + ring_start * d, H, runs.len_a * d, capacity * d);
    cast(kc_s + runs.len_a * d, cache_len * d, kc_f, H, runs.len_b * d, capacity * d);
    cast(vc_s + runs.len_a * d, cache_len * d, vc_f, H, runs.len_b * d, capacity * d);
    cast(kn_b, hd, k_new, Ln, hd, tok_heads * d);
    cast(vn_b, hd, v_new, Ln, hd, tok_heads * d);
    if (launches) wsi::count_launch(launches);
    if (ce != cudaSuccess) return wsi::cuda_fail(ce);
  }
  if (kv8) return d == 128 ? launch_attention<128, false, true>(prm, dev, stream) : launch_attention<64, false, true>(prm, dev, stream);
  // BF16 operands read in place, FP32 rows out (wsi::attn_bf16_in_f32_out): the FP32 epilogue without the staging casts
  if (f32_out_only) return d == 128 ? launch_attention<128, true, false>(prm, dev, stream) : launch_attention<64, true, false>(prm, dev, stream);
  if (d == 128) return f32 ? launch_attention<128, true, false>(prm, dev, stream) : launch_attention<128, false, false>(prm, dev, stream);
  return f32 ? launch_attention<64, true, false>(prm, dev, stream) : launch_attention<64, false, false>(prm, dev, stream);
}
}  // namespace

extern "C" __attribute__((visibility("default"))) int ws_block_causal_attn(void* out, float* lse, const void* q, const void* k_cache, const void* v_cache,
                                    int64_t capacity, int64_t cache_len, const void* k_new, const void* v_new, int32_t Ln,
                                    int32_t H, int32_t d, int32_t Lq, const ws_block_mask* mask, float softmax_scale,
                                    void* workspace, size_t workspace_bytes, ws_dtype dt, void* stream) {
  return attn_impl(out, lse, q, k_cache, v_cache, capacity, cache_len, k_new, v_new, Ln, H, d, Lq, mask, softmax_scale, workspace,
                   workspace_bytes, dt, stream, H);
}

// Internal (ws_unit.cu): ws_block_causal_attn on BF16 inputs whose output rows are written as FP32 [Lq, H, d] -- the
// normalised O before its rounding to BF16, for partial results that are merged afterwards.
int wsi::attn_bf16_in_f32_out(float* out, float* lse, const void* q, const void* k_cache, const void* v_cache, int64_t capacity,
                              int64_t cache_len, const void* k_new, const void* v_new, int32_t Ln, int32_t H, int32_t d, int32_t Lq,
                              const ws_block_mask* mask, float softmax_scale, void* workspace, size_t workspace_bytes, void* stream) {
  return attn_impl(out, lse, q, k_cache, v_cache, capacity, cache_len, k_new, v_new, Ln, H, d, Lq, mask, softmax_scale, workspace,
                   workspace_bytes, WS_DTYPE_BF16, stream, H, nullptr, nullptr, 0, nullptr, 1, 0, true);
}

// a2 + a3 + a4 in one call: the rank's heads [head_begin, head_begin + H) are read straight from
// the token-major [n_tok, H_total, d] tensors by strided TMA and O is stored straight back into that layout.
extern "C" __attribute__((visibility("default"))) int ws_block_causal_attn_seq_layout(void* out_seq, float* lse, const void* q_seq, const void* k_cache,
                                               const void* v_cache, int64_t capacity, int64_t cache_len, const void* k_new_seq,
                                               const void* v_new_seq, int32_t Ln, int32_t H_total, int32_t head_begin, int32_t H,
                                               int32_t d, int32_t Lq, const ws_block_mask* mask, float softmax_scale,
                                               void* workspace, size_t workspace_bytes, ws_dtype dt, void* stream) {
  if (dt != WS_DTYPE_BF16 && dt != WS_DTYPE_F32) return WS_ERR_UNSUPPORTED;
  if (H_total <= 0 || H <= 0 || d <= 0 || head_begin < 0 || (int64_t)head_begin + H > H_total) return WS_ERR_INVALID_ARG;
  const int64_t off = (int64_t)head_begin * d * wsi::elem_bytes(dt);
  auto shift = [off](const void* p) { return p ? static_cast<const void*>(static_cast<const char*>(p) + off) : nullptr; };
  return attn_impl(out_seq ? static_cast<char*>(out_seq) + off : nullptr, lse, shift(q_seq), k_cache, v_cache, capacity, cache_len,
                   shift(k_new_seq), shift(v_new_seq), Ln, H, d, Lq, mask, softmax_scale, workspace, workspace_bytes, dt, stream,
                   H_total);
}

// a3 with exchange #2 of the Ulysses group fused into its epilogue ("Ulysses all-to-all/gather
// communication", :73; R20).  This rank (index `rank` of P) computes its H heads over the whole sequence
// (P * Ls sharded rows, then Lq - P * Ls unsharded rows) and the softmax warps store every finished row straight into
// the token-major [Ls + La, P * H, d] output of the peer that owns the row -- peer i / Ls for a sharded row i, EVERY peer
// for an unsharded row (the all-gather) -- through peer-mapped pointers: the all-to-all is the epilogue's store, nothing is
// staged and nothing is sent twice.
extern "C" __attribute__((visibility("default"))) int ws_block_causal_attn_push_out(void* const* peer_outs, int32_t P, int32_t rank, int64_t Ls, float* lse, const void* q,
                                             const void* k_cache, const void* v_cache, int64_t capacity, int64_t cache_len,
                                             const void* k_new, const void* v_new, int32_t Ln, int32_t H, int32_t d, int32_t Lq,
                                             const ws_block_mask* mask, float softmax_scale, void* workspace, size_t workspace_bytes,
                                             ws_dtype dt, void* stream) {
  if (dt != WS_DTYPE_BF16 && dt != WS_DTYPE_F32) return WS_ERR_UNSUPPORTED;
  if (!peer_outs || P <= 0 || rank < 0 || rank >= P || Ls <= 0 || H <= 0 || d <= 0 || Lq <= 0) return WS_ERR_INVALID_ARG;
  if (P > WS_MAX_PEERS) return WS_ERR_UNSUPPORTED;
  if ((int64_t)P * Ls > Lq) return WS_ERR_OUT_OF_RANGE;
  const int64_t off = (int64_t)rank * H * d * wsi::elem_bytes(dt);  // this rank's first head inside a [*, P * H, d] token row
  void* shifted[WS_MAX_PEERS];
  const size_t peer_bytes = (size_t)(Ls + (Lq - (int64_t)P * Ls)) * P * H * d * wsi::elem_bytes(dt);
  for (int r = 0; r < P; ++r) {
    if (!peer_outs[r]) return WS_ERR_INVALID_ARG;
    if (!wsi::aligned16(peer_outs[r])) return WS_ERR_ALIGNMENT;
    for (int j = 0; j < r; ++j)
      if (wsi::ranges_overlap(peer_outs[r], peer_bytes, peer_outs[j], peer_bytes)) return WS_ERR_OVERLAP;
    shifted[r] = static_cast<char*>(peer_outs[r]) + off;
  }
  // A peer's output may not alias anything this call reads or uses as scratch: the epilogue stores finished rows while
  // other CTAs are still reading Q, K/V and the partial records.  (Sizes of arguments that attn_impl will reject are skipped.)
  const size_t es = (size_t)wsi::elem_bytes(dt);
  const size_t new_bytes = Ln > 0 ? (size_t)Ln * H * d * es : 0, cache_bytes = capacity > 0 ? (size_t)H * capacity * d * es : 0;
  for (int r = 0; r < P; ++r) {
    const void* reads[] = {q, k_new, v_new, k_cache, v_cache, lse, workspace};
    const size_t sizes[] = {(size_t)Lq * H * d * es, new_bytes, new_bytes, cache_bytes, cache_bytes, (size_t)H * Lq * 4, workspace_bytes};
    for (int i = 0; i < 7; ++i)
      if (reads[i] && wsi::ranges_overlap(peer_outs[r], peer_bytes, reads[i], sizes[i])) return WS_ERR_OVERLAP;
  }
  return attn_impl(shifted[0], lse, q, k_cache, v_cache, capacity, cache_len, k_new, v_new, Ln, H, d, Lq, mask, softmax_scale, workspace,
                   workspace_bytes, dt, stream, H, nullptr, nullptr, 0, shifted, P, Ls);
}

// a3 on a ring (sliding-window) cache, SURVEY.md 8(f).4 / DESIGN.md R19: cache key j of the timeline is physical row
// (ring_start + j) mod capacity.  The window is at most two physical runs of the cache tensor; each is tiled on its own.
extern "C" __attribute__((visibility("default"))) int ws_block_causal_attn_ring(void* out, float* lse, const void* q, const void* k_cache, const void* v_cache,
                                         int64_t capacity, int64_t ring_start, int64_t cache_len, const void* k_new, const void* v_new,
                                         int32_t Ln, int32_t H, int32_t d, int32_t Lq, const ws_block_mask* mask, float softmax_scale,
                                         void* workspace, size_t workspace_bytes, ws_dtype dt, void* stream) {
  if (ring_start < 0 || ring_start >= (capacity > 0 ? capacity : 1)) return WS_ERR_OUT_OF_RANGE;
  return attn_impl(out, lse, q, k_cache, v_cache, capacity, cache_len, k_new, v_new, Ln, H, d, Lq, mask, softmax_scale, workspace,
                   workspace_bytes, dt, stream, H, nullptr, nullptr, ring_start);
}

// a3 on an FP8 cache: the cache holds E4M3 codes and one power-of-two exponent per (row, head), written by
// ws_kv_cache_write_fp8; the unit's own K/V stay BF16.  The codes are expanded to BF16 inside the SM, exactly, so the result is
// BF16 attention on the dequantised cache.
extern "C" __attribute__((visibility("default"))) int ws_block_causal_attn_fp8kv(void* out, float* lse, const void* q, const void* k_cache8, const void* v_cache8,
                                          const int8_t* k_exp, const int8_t* v_exp, int64_t capacity, int64_t cache_len,
                                          const void* k_new, const void* v_new, int32_t Ln, int32_t H, int32_t d, int32_t Lq,
                                          const ws_block_mask* mask, float softmax_scale, void* workspace, size_t workspace_bytes,
                                          void* stream) {
  if (!k_exp || !v_exp) return WS_ERR_INVALID_ARG;
  if (capacity % 16 != 0 || (reinterpret_cast<uintptr_t>(k_exp) & 15) || (reinterpret_cast<uintptr_t>(v_exp) & 15)) return WS_ERR_ALIGNMENT;
  // the exponent arrays are read throughout the launch: neither the output nor the scratch may sit on top of them
  if (out && H > 0 && d > 0 && Lq > 0 && capacity > 0) {
    const size_t exp_bytes = (size_t)H * capacity, out_bytes = (size_t)Lq * H * d * 2;
    for (const int8_t* e : {k_exp, v_exp})
      if (wsi::ranges_overlap(e, exp_bytes, out, out_bytes) || (workspace && wsi::ranges_overlap(e, exp_bytes, workspace, workspace_bytes)) ||
          (lse && wsi::ranges_overlap(e, exp_bytes, lse, (size_t)H * Lq * 4)))
        return WS_ERR_OVERLAP;
  }
  return attn_impl(out, lse, q, k_cache8, v_cache8, capacity, cache_len, k_new, v_new, Ln, H, d, Lq, mask, softmax_scale, workspace,
                   workspace_bytes, WS_DTYPE_BF16, stream, H, k_exp, v_exp);
}
