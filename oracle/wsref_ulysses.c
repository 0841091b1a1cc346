/*
 * wsref_ulysses.c -- CPU ORACLE for the Ulysses exchange of the performer group, SURVEY.md 8(f).2
 *                    ("denoising for the long latent video sequence is split across ranks with Ulysses
 *                    all-to-all/gather communication.  Audio latents ... are generated without sequence sharding";
 *                    PAPER.md:65 Table 1 "Thinker broadcasts performer-compatible K/V slices").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (see wsref.c): only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline leg may build, load or call it.  It shares nothing with paper_2607_04443_b200/csrc/.
 *
 * The paper names the collectives and gives no index map; the map below is the standard Ulysses one plus a reading of
 * "all-to-all/gather" for the unsharded audio tokens (R20):
 *
 *   P ranks, H heads, Hp = H / P heads per rank.  A unit's sequence is Ls * P sharded (video) tokens followed by La
 *   unsharded (audio) tokens.  Rank r holds, for all H heads, the token-major tensor
 *       X_r [Ls + La, H, d]:  rows [0, Ls) = video tokens r * Ls .. (r + 1) * Ls - 1, rows [Ls, Ls + La) = the audio
 *       tokens (replicated: every rank holds the same La rows).
 *   Attention is head-parallel: rank g needs, for its heads [g * Hp, (g + 1) * Hp), the whole sequence
 *       Y_g [P * Ls + La, Hp, d].
 *
 *   exchange #1 (all-to-all, before attention; Q, K_new, V_new):
 *       Y_g[r * Ls + t, c, :] = X_r[t, g * Hp + c, :]            0 <= r < P, 0 <= t < Ls, 0 <= c < Hp
 *       Y_g[P * Ls + a, c, :] = X_g[Ls + a, g * Hp + c, :]       0 <= a < La   (local: the audio rows are replicated)
 *   exchange #2 (all-to-all for the video rows, all-GATHER for the audio rows, after attention; O):
 *       Z_r[t, g * Hp + c, :]      = O_g[r * Ls + t, c, :]       0 <= g < P, 0 <= t < Ls, 0 <= c < Hp
 *       Z_r[Ls + a, g * Hp + c, :] = O_g[P * Ls + a, c, :]       0 <= a < La   (every rank receives every head)
 *   K/V-slice broadcast fused with the cache write (a1 on every rank):
 *       cache_g[h, row_offset + i, :] = S[i, g * Hp + h, :]      0 <= g < P, 0 <= h < Hp, 0 <= i < n_rows
 *
 * Pins (tests/test_oracle_ulysses_pins.py, no GPU): numpy reshape / transpose / concatenate statements of the same maps,
 * #2 o #1 = identity on every rank, element-id tensors, the composition "exchange #1 -> per-rank attention on Hp heads ->
 * exchange #2" against single-rank attention on all H heads (heads are independent), the broadcast write against
 * wsref_kv_cache_write per rank, and the two exchanges carried out for real by torch.distributed (gloo, 2 and 4 CPU
 * ranks: all_to_all_single + all_gather).  No function here is "parity unpinned".
 *
 * Build:  gcc -O2 -fPIC -shared -o libwsref_ulysses.so wsref_ulysses.c
 */
#include <stdint.h>

#define WSREF_OK 0
#define WSREF_BAD_ARG (-1)

/* Y_g from the P tensors X_0 .. X_{P-1} (x[r] points to X_r). */
int wsref_ulysses_seq_to_head(uint8_t* y_g, const uint8_t* const* x, int32_t g, int32_t P, int64_t Ls, int64_t La, int32_t H,
                              int32_t d, int32_t elem_bytes) {
  if (P <= 0 || H <= 0 || H % P != 0 || g < 0 || g >= P || Ls < 0 || La < 0 || d <= 0) return WSREF_BAD_ARG;
  const int32_t Hp = H / P;
  const int64_t row = (int64_t)d * elem_bytes;
  for (int32_t r = 0; r < P; ++r)
    for (int64_t t = 0; t < Ls; ++t)
      for (int32_t c = 0; c < Hp; ++c)
        for (int64_t b = 0; b < row; ++b) y_g[((r * Ls + t) * Hp + c) * row + b] = x[r][(t * H + (int64_t)g * Hp + c) * row + b];
  for (int64_t a = 0; a < La; ++a)
    for (int32_t c = 0; c < Hp; ++c)
      for (int64_t b = 0; b < row; ++b) y_g[((P * Ls + a) * Hp + c) * row + b] = x[g][((Ls + a) * H + (int64_t)g * Hp + c) * row + b];
  return WSREF_OK;
}

/* Z_r from the P tensors O_0 .. O_{P-1} (o[g] points to O_g). */
int wsref_ulysses_head_to_seq(uint8_t* z_r, const uint8_t* const* o, int32_t r, int32_t P, int64_t Ls, int64_t La, int32_t H,
                              int32_t d, int32_t elem_bytes) {
  if (P <= 0 || H <= 0 || H % P != 0 || r < 0 || r >= P || Ls < 0 || La < 0 || d <= 0) return WSREF_BAD_ARG;
  const int32_t Hp = H / P;
  const int64_t row = (int64_t)d * elem_bytes;
  for (int32_t g = 0; g < P; ++g) {
    for (int64_t t = 0; t < Ls; ++t)
      for (int32_t c = 0; c < Hp; ++c)
        for (int64_t b = 0; b < row; ++b) z_r[(t * H + (int64_t)g * Hp + c) * row + b] = o[g][((r * Ls + t) * Hp + c) * row + b];
    for (int64_t a = 0; a < La; ++a)
      for (int32_t c = 0; c < Hp; ++c)
        for (int64_t b = 0; b < row; ++b)
          z_r[((Ls + a) * H + (int64_t)g * Hp + c) * row + b] = o[g][((P * Ls + a) * Hp + c) * row + b];
  }
  return WSREF_OK;
}

/* The thinker's slice S [n_rows, P * Hp, d] written into every rank's cache [Hp, capacity, d] (k_caches[g], v_caches[g]). */
int wsref_kv_slice_broadcast_write(uint8_t* const* k_caches, uint8_t* const* v_caches, int32_t P, int64_t capacity, int32_t Hp,
                                   int32_t d, const uint8_t* k_src, const uint8_t* v_src, int32_t n_rows, int64_t row_offset,
                                   int32_t elem_bytes) {
  if (P <= 0 || Hp <= 0 || d <= 0 || n_rows < 0 || row_offset < 0 || row_offset + n_rows > capacity) return WSREF_BAD_ARG;
  const int64_t row = (int64_t)d * elem_bytes;
  const int64_t H = (int64_t)P * Hp;
  for (int32_t g = 0; g < P; ++g)
    for (int32_t h = 0; h < Hp; ++h)
      for (int32_t i = 0; i < n_rows; ++i)
        for (int64_t b = 0; b < row; ++b) {
          const int64_t dst = (((int64_t)h * capacity) + row_offset + i) * row + b;
          const int64_t src = (((int64_t)i * H) + (int64_t)g * Hp + h) * row + b;
          k_caches[g][dst] = k_src[src];
          v_caches[g][dst] = v_src[src];
        }
  return WSREF_OK;
}
