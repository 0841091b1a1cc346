/*
 * wsref.c -- CPU ORACLE for the Wan-Streamer v0.2 performer hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may build, load or call it.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_2607_04443_b200/csrc/ and includes nothing from include/.
 *
 * What it computes (PAPER.md line numbers; the paper gives names and data flow,
 * no equations, so each function is the plain textbook definition -- see
 * DESIGN.md "Readings" R1..R16 for every place the paper is silent):
 *
 *   wsref_kv_cache_write   PAPER.md:11,:31,:79  "each performer rank writes incoming
 *                          K/V into a pre-sharded local cache"          -> index map
 *   wsref_seq_to_head /    PAPER.md:31,:73 "Ulysses all-to-all/gather collectives
 *   wsref_head_to_seq      around attention" -- the rank-local halves   -> index map
 *   wsref_block_causal_attn PAPER.md:25 "coordinated by block-causal attention"
 *                          -> masked softmax attention, by definition, in FP64
 *
 * Plain loops, no blocking, no online softmax, no reordering: for every query row
 * the scores of all visible keys are formed, the maximum is subtracted, the
 * exponentials are summed and the weighted mean of the value rows is taken.
 *
 * Pins (tests/test_oracle_pins.py, all run without a GPU): brute-force pure-Python
 * definition on tiny inputs, the numpy explicit-mask twin (oracle/dense_twin.py,
 * separate code), torch FP64 scaled_dot_product_attention, closed forms (equal keys
 * -> mean of V, one visible key -> v_0, one-hot keys), invariants (row sum 1,
 * permutation within a block, key shift, V linearity, merge identity), the
 * hand-worked fixture tests/golden/softmax_two_keys.txt; relayout/cache-write
 * against numpy transpose / slicing and round trips.  No function here is
 * "parity unpinned".
 *
 * Build:  gcc -O2 -fopenmp -fPIC -shared -o libwsref.so wsref.c -lm     (no -ffast-math)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define WSREF_OK 0
#define WSREF_BAD_ARG (-1)

int wsref_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------------
 * a1. KV cache write ("each performer rank writes them into its pre-sharded
 *     local cache"; R5: the shard is a head range, the cache is head-major).
 *
 *     cache[h, row_offset + r, c] = src[r, head_begin + h, c]      for K and for V,
 *     0 <= h < H, 0 <= r < n_rows, 0 <= c < d; every other cache byte is left alone.
 *     cache: [H, capacity, d]   src: [n_rows, H_src, d]   elements of elem_bytes bytes.
 * ---------------------------------------------------------------------------------------- */
int wsref_kv_cache_write(uint8_t* k_cache, uint8_t* v_cache, int64_t capacity, int32_t H, int32_t d,
                         const uint8_t* k_src, const uint8_t* v_src, int32_t n_rows, int32_t H_src,
                         int32_t head_begin, int64_t row_offset, int32_t elem_bytes) {
  if (H <= 0 || d <= 0 || n_rows < 0 || H_src <= 0 || head_begin < 0 || head_begin + H > H_src) return WSREF_BAD_ARG;
  if (row_offset < 0 || row_offset + n_rows > capacity) return WSREF_BAD_ARG;
  for (int32_t h = 0; h < H; ++h)
    for (int32_t r = 0; r < n_rows; ++r)
      for (int32_t c = 0; c < d; ++c)
        for (int32_t e = 0; e < elem_bytes; ++e) {
          int64_t dst = ((((int64_t)h * capacity) + row_offset + r) * d + c) * elem_bytes + e;
          int64_t src = ((((int64_t)r * H_src) + head_begin + h) * d + c) * elem_bytes + e;
          k_cache[dst] = k_src[src];
          v_cache[dst] = v_src[src];
        }
  return WSREF_OK;
}

/* ------------------------------------------------------------------------------------------
 * a2. seq->head relayout: the rank-local pack before Ulysses all-to-all #1.
 *     Hp = H / P heads per group.
 *     dst[g, t, c, :] = src[t, (g0 + g) * Hp + c, :]     0<=g<G, 0<=t<n_tok, 0<=c<Hp
 *     src: [n_tok, H, d]    dst: [G, n_tok, Hp, d]
 * ---------------------------------------------------------------------------------------- */
int wsref_seq_to_head(uint8_t* dst, const uint8_t* src, int64_t n_tok, int32_t H, int32_t d, int32_t P,
                      int32_t g0, int32_t G, int32_t elem_bytes) {
  if (P <= 0 || H % P != 0 || g0 < 0 || G < 0 || g0 + G > P) return WSREF_BAD_ARG;
  const int32_t Hp = H / P;
  const int64_t row = (int64_t)d * elem_bytes;
  for (int32_t g = 0; g < G; ++g)
    for (int64_t t = 0; t < n_tok; ++t)
      for (int32_t c = 0; c < Hp; ++c)
        for (int64_t b = 0; b < row; ++b)
          dst[(((int64_t)g * n_tok + t) * Hp + c) * row + b] = src[(t * H + (int64_t)(g0 + g) * Hp + c) * row + b];
  return WSREF_OK;
}

/* a4. head->seq relayout: the rank-local unpack after all-to-all #2; inverse of a2.
 *     dst[t, (g0 + g) * Hp + c, :] = src[g, t, c, :]; heads outside the G groups untouched. */
int wsref_head_to_seq(uint8_t* dst, const uint8_t* src, int64_t n_tok, int32_t H, int32_t d, int32_t P,
                      int32_t g0, int32_t G, int32_t elem_bytes) {
  if (P <= 0 || H % P != 0 || g0 < 0 || G < 0 || g0 + G > P) return WSREF_BAD_ARG;
  const int32_t Hp = H / P;
  const int64_t row = (int64_t)d * elem_bytes;
  for (int32_t g = 0; g < G; ++g)
    for (int64_t t = 0; t < n_tok; ++t)
      for (int32_t c = 0; c < Hp; ++c)
        for (int64_t b = 0; b < row; ++b)
          dst[(t * H + (int64_t)(g0 + g) * Hp + c) * row + b] = src[(((int64_t)g * n_tok + t) * Hp + c) * row + b];
  return WSREF_OK;
}

/* ------------------------------------------------------------------------------------------
 * a3. Block-causal unit attention (R1, R2, R11, R16).
 *
 * Key timeline: index j < cache_len is cache row j; cache_len <= j < cache_len + Ln is row
 * j - cache_len of the unit's own ("new") K/V.  Query row i lies in block b(i), the first
 * block with i < q_block_end[b]; it sees exactly the keys j < kv_visible[b(i)].
 *
 *     s_j  = softmax_scale * sum_c q[i,h,c] * k_j[h,c]                (c ascending, double)
 *     m    = max_j s_j ;  p_j = exp(s_j - m) ;  l = sum_j p_j         (j ascending)
 *     O[i,h,c] = (sum_j p_j * v_j[h,c]) / l ;   lse[h,i] = m + log(l)
 *     no visible key  ->  O = 0, lse = -inf                            (R11)
 *
 * Inputs are float32 arrays holding the exact values the GPU receives (BF16 values are
 * exactly representable in float32); all arithmetic is double.
 *   q, k_new, v_new : [L, H, d] token-major     k_cache, v_cache : [H, capacity, d]
 * ---------------------------------------------------------------------------------------- */
typedef struct {
  const float *q, *k_cache, *v_cache, *k_new, *v_new;
  int64_t capacity, cache_len;
  int32_t Ln, H, d, Lq, n_blocks;
  const int32_t *q_block_end, *kv_visible;
  double scale;
} attn_problem;

static int32_t block_of_row(const attn_problem* p, int32_t i) {
  for (int32_t b = 0; b < p->n_blocks; ++b)
    if (i < p->q_block_end[b]) return b;
  return -1;
}

static const float* key_row(const attn_problem* p, int32_t h, int64_t j) {
  if (j < p->cache_len) return p->k_cache + ((int64_t)h * p->capacity + j) * p->d;
  return p->k_new + ((j - p->cache_len) * p->H + h) * p->d;
}

static const float* value_row(const attn_problem* p, int32_t h, int64_t j) {
  if (j < p->cache_len) return p->v_cache + ((int64_t)h * p->capacity + j) * p->d;
  return p->v_new + ((j - p->cache_len) * p->H + h) * p->d;
}

/* one (row, head): writes d outputs, one lse, and (if p_row != NULL) the n normalised weights */
static void attend_row(const attn_problem* p, int32_t i, int32_t h, double* scores, double* out_row, double* lse_out,
                       double* p_row) {
  const int32_t d = p->d;
  const int32_t b = block_of_row(p, i);
  const int64_t n = p->kv_visible[b];
  if (n == 0) {
    for (int32_t c = 0; c < d; ++c) out_row[c] = 0.0;
    *lse_out = -INFINITY;
    return;
  }
  const float* qi = p->q + ((int64_t)i * p->H + h) * d;
  double m = -INFINITY;
  for (int64_t j = 0; j < n; ++j) {
    const float* kj = key_row(p, h, j);
    double acc = 0.0;
    for (int32_t c = 0; c < d; ++c) acc += (double)qi[c] * (double)kj[c];
    scores[j] = p->scale * acc;
    if (scores[j] > m) m = scores[j];
  }
  double l = 0.0;
  for (int64_t j = 0; j < n; ++j) {
    scores[j] = exp(scores[j] - m);
    l += scores[j];
  }
  for (int32_t c = 0; c < d; ++c) out_row[c] = 0.0;
  for (int64_t j = 0; j < n; ++j) {
    const float* vj = value_row(p, h, j);
    const double w = scores[j];
    for (int32_t c = 0; c < d; ++c) out_row[c] += w * (double)vj[c];
  }
  for (int32_t c = 0; c < d; ++c) out_row[c] /= l;
  *lse_out = m + log(l);
  if (p_row)
    for (int64_t j = 0; j < n; ++j) p_row[j] = scores[j] / l;
}

static int check_problem(const attn_problem* p) {
  if (p->H <= 0 || p->d <= 0 || p->Lq < 0 || p->Ln < 0 || p->n_blocks <= 0) return WSREF_BAD_ARG;
  if (p->cache_len < 0 || p->cache_len > p->capacity) return WSREF_BAD_ARG;
  int32_t prev_end = 0, prev_vis = 0;
  for (int32_t b = 0; b < p->n_blocks; ++b) {
    if (p->q_block_end[b] <= prev_end) return WSREF_BAD_ARG;
    if (p->kv_visible[b] < prev_vis || (int64_t)p->kv_visible[b] > p->cache_len + p->Ln) return WSREF_BAD_ARG;
    prev_end = p->q_block_end[b];
    prev_vis = p->kv_visible[b];
  }
  if (prev_end != p->Lq) return WSREF_BAD_ARG;
  return WSREF_OK;
}

/* out: [Lq, H, d] double; lse: [H, Lq] double (may be NULL);
 * p_rows: NULL, or [H, Lq, cache_len + Ln] double receiving the normalised weights (0 beyond the visible prefix). */
int wsref_block_causal_attn(double* out, double* lse, const float* q, const float* k_cache, const float* v_cache,
                            int64_t capacity, int64_t cache_len, const float* k_new, const float* v_new, int32_t Ln,
                            int32_t H, int32_t d, int32_t Lq, int32_t n_blocks, const int32_t* q_block_end,
                            const int32_t* kv_visible, double softmax_scale, double* p_rows) {
  attn_problem p = {q, k_cache, v_cache, k_new, v_new, capacity, cache_len, Ln, H, d, Lq, n_blocks, q_block_end, kv_visible,
                    softmax_scale};
  int rc = check_problem(&p);
  if (rc != WSREF_OK) return rc;
  const int64_t kv_total = cache_len + Ln;
  const int64_t n_items = (int64_t)H * Lq;
  int failed = 0;
#pragma omp parallel
  {
    double* scores = (double*)malloc(sizeof(double) * (size_t)(kv_total > 0 ? kv_total : 1));
    if (!scores) {
#pragma omp atomic write
      failed = 1;
    }
#pragma omp for schedule(dynamic, 8)
    for (int64_t it = 0; it < n_items; ++it) {
      if (!scores) continue;
      const int32_t h = (int32_t)(it / Lq), i = (int32_t)(it % Lq);
      double lse_v;
      double* prow = NULL;
      if (p_rows) {
        prow = p_rows + ((int64_t)h * Lq + i) * kv_total;
        for (int64_t j = 0; j < kv_total; ++j) prow[j] = 0.0;
      }
      attend_row(&p, i, h, scores, out + ((int64_t)i * H + h) * d, &lse_v, prow);
      if (lse) lse[(int64_t)h * Lq + i] = lse_v;
    }
    free(scores);
  }
  return failed ? WSREF_BAD_ARG : WSREF_OK;
}

/* The same definition on a list of (row, head) samples only -- rows are independent, so a
 * sample is exact for those rows.  out: [n_samples, d]; lse: [n_samples] (may be NULL). */
int wsref_block_causal_attn_rows(double* out, double* lse, const float* q, const float* k_cache, const float* v_cache,
                                 int64_t capacity, int64_t cache_len, const float* k_new, const float* v_new, int32_t Ln,
                                 int32_t H, int32_t d, int32_t Lq, int32_t n_blocks, const int32_t* q_block_end,
                                 const int32_t* kv_visible, double softmax_scale, int32_t n_samples,
                                 const int32_t* sample_rows, const int32_t* sample_heads) {
  attn_problem p = {q, k_cache, v_cache, k_new, v_new, capacity, cache_len, Ln, H, d, Lq, n_blocks, q_block_end, kv_visible,
                    softmax_scale};
  int rc = check_problem(&p);
  if (rc != WSREF_OK) return rc;
  for (int32_t s = 0; s < n_samples; ++s)
    if (sample_rows[s] < 0 || sample_rows[s] >= Lq || sample_heads[s] < 0 || sample_heads[s] >= H) return WSREF_BAD_ARG;
  const int64_t kv_total = cache_len + Ln;
  int failed = 0;
#pragma omp parallel
  {
    double* scores = (double*)malloc(sizeof(double) * (size_t)(kv_total > 0 ? kv_total : 1));
    if (!scores) {
#pragma omp atomic write
      failed = 1;
    }
#pragma omp for schedule(dynamic, 1)
    for (int32_t s = 0; s < n_samples; ++s) {
      if (!scores) continue;
      double lse_v;
      attend_row(&p, sample_rows[s], sample_heads[s], scores, out + (int64_t)s * d, &lse_v, NULL);
      if (lse) lse[s] = lse_v;
    }
    free(scores);
  }
  return failed ? WSREF_BAD_ARG : WSREF_OK;
}
