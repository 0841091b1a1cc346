/*
 * wsref_ring.c -- CPU ORACLE for the sliding-window (ring-buffer) K/V cache, SURVEY.md 8(f).4
 *                 ("cache windowing/eviction for unbounded sessions"; "full-history cache",
 *                 PAPER.md:47 one committed unit per 160 ms, without end).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (see wsref.c): only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline leg may build, load or call it.  It shares nothing with paper_2607_04443_b200/csrc/.
 *
 * The paper gives no eviction rule, so the rule is a reading (R19):
 *
 *   The cache is a ring of `capacity` rows per head that keeps the MOST RECENT rows of the session.  Rows are numbered
 *   by their position in the session, w = 0, 1, 2, ... (the "write position"); row w lives in physical row w mod capacity
 *   and stays there until row w + capacity overwrites it (first in, first out).
 *
 *   After W rows have been written the window holds the rows max(0, W - capacity) .. W - 1:
 *       cache_len  = min(W, capacity)                          valid rows
 *       ring_start = W < capacity ? 0 : W mod capacity         physical row of the OLDEST valid row
 *   and key j of the attention timeline (0 <= j < cache_len, oldest first) is physical row (ring_start + j) mod capacity.
 *   Attention on a ring cache is, by definition, wsref_block_causal_attn on the linearised window (wsref_ring_linearise);
 *   the Python front end does exactly that.
 *
 * Pins (tests/test_oracle_ring_pins.py, no GPU): the write against numpy fancy indexing with `% capacity`, against the
 * linear wsref_kv_cache_write when nothing wraps, and a session of many writes against "keep the last `capacity` rows
 * of the concatenation"; the linearisation against numpy.roll; the state rule against a brute-force simulation; ring
 * attention with a fully visible cache against attention on the physical order (softmax is invariant under a
 * permutation of the keys) and a spike key on each side of the wrap seam.  No function here is "parity unpinned".
 *
 * Build:  gcc -O2 -fPIC -shared -o libwsref_ring.so wsref_ring.c
 */
#include <stdint.h>

#define WSREF_OK 0
#define WSREF_BAD_ARG (-1)

/* The window after W rows of the session have been written (see the header). */
int wsref_ring_state(int64_t W, int64_t capacity, int64_t* ring_start, int64_t* cache_len) {
  if (W < 0 || capacity <= 0) return WSREF_BAD_ARG;
  if (W < capacity) {
    *ring_start = 0;
    *cache_len = W;
  } else {
    *ring_start = W % capacity;
    *cache_len = capacity;
  }
  return WSREF_OK;
}

/*   cache[h, (write_pos + r) mod capacity, c] = src[r, head_begin + h, c]      for K and for V,
 *   0 <= h < H, 0 <= r < n_rows, 0 <= c < d; every other cache byte is left alone.
 *   cache: [H, capacity, d]   src: [n_rows, H_src, d]   elements of elem_bytes bytes.
 *   n_rows <= capacity: a call never overwrites a row it has written itself. */
int wsref_kv_cache_write_ring(uint8_t* k_cache, uint8_t* v_cache, int64_t capacity, int32_t H, int32_t d,
                              const uint8_t* k_src, const uint8_t* v_src, int32_t n_rows, int32_t H_src, int32_t head_begin,
                              int64_t write_pos, int32_t elem_bytes) {
  if (H <= 0 || d <= 0 || n_rows < 0 || H_src <= 0 || head_begin < 0 || head_begin + H > H_src) return WSREF_BAD_ARG;
  if (capacity <= 0 || write_pos < 0 || n_rows > capacity) return WSREF_BAD_ARG;
  for (int32_t h = 0; h < H; ++h)
    for (int32_t r = 0; r < n_rows; ++r) {
      const int64_t phys = (write_pos + r) % capacity;
      for (int32_t c = 0; c < d; ++c)
        for (int32_t e = 0; e < elem_bytes; ++e) {
          const int64_t dst = ((((int64_t)h * capacity) + phys) * d + c) * elem_bytes + e;
          const int64_t src = ((((int64_t)r * H_src) + head_begin + h) * d + c) * elem_bytes + e;
          k_cache[dst] = k_src[src];
          v_cache[dst] = v_src[src];
        }
    }
  return WSREF_OK;
}

/*   lin[h, j, :] = cache[h, (ring_start + j) mod capacity, :]     0 <= j < cache_len <= capacity
 *   lin: [H, cache_len, d]   cache: [H, capacity, d] */
int wsref_ring_linearise(uint8_t* lin, const uint8_t* cache, int64_t capacity, int32_t H, int32_t d, int64_t ring_start,
                         int64_t cache_len, int32_t elem_bytes) {
  if (H <= 0 || d <= 0 || capacity <= 0 || ring_start < 0 || ring_start >= capacity || cache_len < 0 || cache_len > capacity)
    return WSREF_BAD_ARG;
  const int64_t row = (int64_t)d * elem_bytes;
  for (int32_t h = 0; h < H; ++h)
    for (int64_t j = 0; j < cache_len; ++j) {
      const int64_t phys = (ring_start + j) % capacity;
      for (int64_t b = 0; b < row; ++b) lin[((int64_t)h * cache_len + j) * row + b] = cache[((int64_t)h * capacity + phys) * row + b];
    }
  return WSREF_OK;
}
