/*
 * wsref_fp8.c -- CPU ORACLE for the FP8 K/V cache row of the hot path (SURVEY.md 8(f).3:
 *                "FP8 K/V cache written by a1 with per-row/head scales", "local shards of
 *                the full-history cache").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as wsref.c: only tests/, smoke() and
 * bench.py's cpu_baseline leg may build, load or call it; it shares nothing with csrc/ or include/).
 *
 * The paper does not describe a quantised cache; the format below is this repository's reading
 * (R17/R18), written out as plain arithmetic in double precision:
 *
 *   element format  OCP FP8 E4M3 ("e4m3fn"): 1 sign, 4 exponent (bias 7), 3 mantissa bits; no infinity;
 *                   S.1111.111 is NaN; exponent field 0 is subnormal: (-1)^s 2^-6 (m/8); otherwise
 *                   (-1)^s 2^(E-7) (1 + m/8); largest finite value 448.
 *   scale           one power of two 2^e per (row, head), e stored as int8:
 *                   e = the smallest integer with 448 * 2^e >= amax, amax = max_c |x[c]| over the d elements
 *                   of the row, clamped to [-100, 7]  (amax == 0 -> e = -100).
 *   code            RN-even(x / 2^e) to E4M3, saturated to +-448 (reached only when e was clamped at 7).
 *   dequantised     decode(code) * 2^e  -- 4 significant bits and an exponent inside BF16's range, hence exactly
 *                   representable in BF16: attention on an FP8 cache IS BF16 attention on the dequantised cache.
 *
 *   wsref_kv_cache_write_fp8: cache8[h, row_offset + r, :], exp[h, row_offset + r] = quantise(src[r, head_begin + h, :])
 *   wsref_kv_cache_dequant_fp8: out[h, r, c] = decode(cache8[h, r, c]) * 2^exp[h, r]
 *
 * Pins (tests/test_oracle_fp8_pins.py, no GPU): the decode table of all 256 codes against torch.float8_e4m3fn,
 * the encoder against torch's float -> float8_e4m3fn conversion and against a brute-force nearest-code search over
 * the decode table (ties to the even code), hand-worked ties / subnormals / saturation, the scale rule at its
 * boundaries, the round-trip error bound, exact BF16 representability, and the index map against numpy slicing.
 *
 * Build:  gcc -O2 -fPIC -shared -o libwsref_fp8.so wsref_fp8.c -lm     (no -ffast-math)
 */
#include <math.h>
#include <stdint.h>

#define WSREF_OK 0
#define WSREF_BAD_ARG (-1)

/* value of an E4M3 code, by the definition of the format (NaN codes return NaN) */
double wsref_e4m3_decode(uint8_t code) {
  const int s = code >> 7, E = (code >> 3) & 15, m = code & 7;
  double v;
  if (E == 15 && m == 7) return NAN;
  if (E == 0) v = ldexp((double)m / 8.0, -6);
  else v = ldexp(1.0 + (double)m / 8.0, E - 7);
  return s ? -v : v;
}

/* nearest E4M3 code to y, ties to even mantissa, magnitudes above 448 saturate to 448; NaN -> 0x7f */
uint8_t wsref_e4m3_encode(double y) {
  if (isnan(y)) return 0x7f;
  const uint8_t sign = signbit(y) ? 0x80 : 0x00;
  const double a = fabs(y);
  if (a > 448.0) return sign | 0x7e;              /* saturate: 448 = 1.110b * 2^8 */
  if (a < ldexp(1.0, -6)) {                        /* subnormal range: multiples of 2^-9 */
    const int q = (int)rint(ldexp(a, 9));          /* rint: round half to even (default rounding mode) */
    return sign | (uint8_t)q;                      /* q == 8 is the smallest normal, code 0x08: same bit pattern */
  }
  int ex;
  (void)frexp(a, &ex);                             /* a = f * 2^ex, f in [0.5, 1)  ->  a in [2^(ex-1), 2^ex) */
  int k = ex - 1;                                  /* a = 2^k * (1.xxx) */
  int q = (int)rint(ldexp(a, 3 - k));              /* in [8, 16] */
  if (q == 16) { q = 8; ++k; }
  return sign | (uint8_t)(((k + 7) << 3) | (q - 8));
}

/* the scale exponent of one row: smallest e with 448 * 2^e >= amax, clamped to [-100, 7] */
int wsref_fp8_row_exponent(const float* x, int32_t d) {
  double amax = 0.0;
  for (int32_t c = 0; c < d; ++c) amax = fmax(amax, fabs((double)x[c]));
  if (amax == 0.0) return -100;
  int e = -100;
  while (e < 7 && ldexp(448.0, e) < amax) ++e;
  return e;
}

/* a1 with quantisation.  cache8: uint8 [H, capacity, d]; exp: int8 [H, capacity]; src: float [n_rows, H_src, d]. */
int wsref_kv_cache_write_fp8(uint8_t* k_cache8, uint8_t* v_cache8, int8_t* k_exp, int8_t* v_exp, int64_t capacity, int32_t H,
                             int32_t d, const float* k_src, const float* v_src, int32_t n_rows, int32_t H_src, int32_t head_begin,
                             int64_t row_offset) {
  if (!k_cache8 || !v_cache8 || !k_exp || !v_exp || capacity <= 0 || H <= 0 || d <= 0 || n_rows < 0 || H_src <= 0 ||
      head_begin < 0 || head_begin + H > H_src || row_offset < 0 || row_offset + n_rows > capacity)
    return WSREF_BAD_ARG;
  if (n_rows > 0 && (!k_src || !v_src)) return WSREF_BAD_ARG;
  for (int which = 0; which < 2; ++which) {
    uint8_t* cache = which ? v_cache8 : k_cache8;
    int8_t* ex = which ? v_exp : k_exp;
    const float* src = which ? v_src : k_src;
    for (int32_t h = 0; h < H; ++h)
      for (int32_t r = 0; r < n_rows; ++r) {
        const float* x = src + ((int64_t)r * H_src + head_begin + h) * d;
        const int e = wsref_fp8_row_exponent(x, d);
        ex[(int64_t)h * capacity + row_offset + r] = (int8_t)e;
        for (int32_t c = 0; c < d; ++c)
          cache[((int64_t)h * capacity + row_offset + r) * d + c] = wsref_e4m3_encode(ldexp((double)x[c], -e));
      }
  }
  return WSREF_OK;
}

/* out[h, r, c] = decode(cache8[h, r, c]) * 2^exp[h, r] for rows [0, n_rows) of every head */
int wsref_kv_cache_dequant_fp8(float* out, const uint8_t* cache8, const int8_t* exp, int64_t capacity, int32_t H, int32_t d,
                               int64_t n_rows) {
  if (!out || !cache8 || !exp || capacity <= 0 || H <= 0 || d <= 0 || n_rows < 0 || n_rows > capacity) return WSREF_BAD_ARG;
  for (int32_t h = 0; h < H; ++h)
    for (int64_t r = 0; r < n_rows; ++r)
      for (int32_t c = 0; c < d; ++c)
        out[((int64_t)h * capacity + r) * d + c] =
            (float)ldexp(wsref_e4m3_decode(cache8[((int64_t)h * capacity + r) * d + c]), exp[(int64_t)h * capacity + r]);
  return WSREF_OK;
}
