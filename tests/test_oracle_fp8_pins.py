"""Pins for the FP8 K/V-cache oracle (oracle/wsref_fp8.c) against things other than itself.  No GPU needed.

The element format is OCP FP8 E4M3, so an independent library routine exists (torch.float8_e4m3fn); the encoder is
additionally pinned by a brute-force nearest-code search (a different algorithm) and by hand-worked cases; the scale
rule and the index map are pinned at their boundaries and against numpy slicing.  DESIGN.md readings R17/R18."""
import math

import numpy as np
import pytest

from oracle import wsref_fp8 as fp8
from paper_2607_04443_b200 import workloads as wl

torch = pytest.importorskip("torch")


def all_codes_decoded():
    return np.array([fp8.e4m3_decode(c) for c in range(256)])


def test_decode_table_matches_torch_float8_e4m3fn_for_all_256_codes():
    ours = all_codes_decoded()
    theirs = torch.arange(256, dtype=torch.uint8).view(torch.float8_e4m3fn).to(torch.float32).numpy().astype(np.float64)
    assert np.array_equal(np.isnan(ours), np.isnan(theirs)) and np.isnan(ours).sum() == 2      # 0x7f and 0xff
    ok = ~np.isnan(ours)
    assert np.array_equal(ours[ok], theirs[ok])
    # and the closed form at the corners of the format
    assert ours[0x7E] == 448.0 and ours[0xFE] == -448.0 and ours[0x08] == 2.0 ** -6 and ours[0x01] == 2.0 ** -9
    assert ours[0x00] == 0.0 and ours[0x38] == 1.0 and ours[0x3C] == 1.5 and ours[0x07] == 7 * 2.0 ** -9


def test_encoder_matches_torch_conversion_inside_the_finite_range():
    rng = np.random.default_rng(1)
    x = np.concatenate([rng.standard_normal(20000) * 3, rng.standard_normal(20000) * 100, rng.uniform(-448, 448, 20000),
                        rng.uniform(-2.0 ** -5, 2.0 ** -5, 20000), all_codes_decoded()[~np.isnan(all_codes_decoded())]]).astype(np.float32)
    x = x[np.abs(x) <= 448.0]
    want = torch.from_numpy(x).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    got = np.array([fp8.e4m3_encode(float(v)) for v in x], np.uint8)
    # torch keeps -0.0 as 0x80 exactly like the oracle (sign of the input)
    assert np.array_equal(got, want)


def test_encoder_matches_brute_force_nearest_code_with_ties_to_even():
    table = all_codes_decoded()
    pos = [(table[c], c) for c in range(0x7F)]            # non-negative finite codes 0x00 .. 0x7e, increasing in value
    vals = np.array([v for v, _ in pos])
    rng = np.random.default_rng(2)
    xs = np.concatenate([rng.uniform(0, 448, 4000), rng.uniform(0, 2.0 ** -5, 2000),
                         (vals[:-1] + vals[1:]) / 2,                     # every exact tie between neighbouring codes
                         np.nextafter((vals[:-1] + vals[1:]) / 2, 0), np.nextafter((vals[:-1] + vals[1:]) / 2, 1e9)])
    for x in xs:
        d = np.abs(vals - x)
        best = np.flatnonzero(d == d.min())
        code = best[0] if len(best) == 1 else [c for c in best if c % 2 == 0][0]   # even mantissa LSB == even code
        assert fp8.e4m3_encode(float(x)) == code, x
        assert fp8.e4m3_encode(float(-x)) == (code | 0x80), -x


def test_hand_worked_ties_subnormals_and_saturation():
    enc, dec = fp8.e4m3_encode, fp8.e4m3_decode
    assert dec(enc(17.0)) == 16.0          # 17 is half way between 16 (mantissa 000) and 18 (001): to even
    assert dec(enc(19.0)) == 20.0          # between 18 (001) and 20 (010)
    assert dec(enc(2.0 ** -10)) == 0.0     # half of the smallest subnormal: to even (zero)
    assert dec(enc(3 * 2.0 ** -10)) == 2.0 ** -8
    assert dec(enc(15.5 * 2.0 ** -10)) == 2.0 ** -6      # rounds up across the subnormal / normal seam
    assert dec(enc(447.9)) == 448.0 and dec(enc(431.9)) == 416.0 and dec(enc(432.0)) == 448.0  # 432: tie 416 (101) / 448 (110)
    assert dec(enc(1000.0)) == 448.0 and dec(enc(-1e30)) == -448.0 and enc(448.0001) == 0x7E   # saturation, never NaN
    assert enc(float("nan")) == 0x7F
    assert enc(-0.0) == 0x80 and enc(0.0) == 0x00


def test_row_exponent_rule_at_its_boundaries():
    row = lambda amax: np.array([amax / 2, -amax, amax / 4, amax / 3], np.float32)
    assert fp8.row_exponent(row(448.0)) == 0
    assert fp8.row_exponent(row(449.0)) == 1 and fp8.row_exponent(row(896.0)) == 1 and fp8.row_exponent(row(897.0)) == 2
    assert fp8.row_exponent(row(224.0)) == -1 and fp8.row_exponent(row(225.0)) == 0
    assert fp8.row_exponent(row(1.0)) == -8 and fp8.row_exponent(row(1.75)) == -8 and fp8.row_exponent(row(1.7578125)) == -7
    assert fp8.row_exponent(np.zeros(8, np.float32)) == -100
    assert fp8.row_exponent(row(1e-37)) == -100                    # lower clamp
    assert fp8.row_exponent(row(57344.0)) == 7 and fp8.row_exponent(row(1e9)) == 7   # upper clamp (then codes saturate)
    # the smallest e with 448 * 2^e >= amax, for random rows
    rng = np.random.default_rng(3)
    for _ in range(300):
        x = (rng.standard_normal(16) * 10.0 ** rng.uniform(-3, 3)).astype(np.float32)
        e, amax = fp8.row_exponent(x), float(np.abs(x).max())
        assert 448.0 * 2.0 ** e >= amax and (e == -100 or 448.0 * 2.0 ** (e - 1) < amax)


def quantise(k, v, H, cap, head_begin, off):
    kc8, vc8 = np.full((H, cap, k.shape[2]), 0xAB, np.uint8), np.full((H, cap, k.shape[2]), 0xCD, np.uint8)
    ke, ve = np.full((H, cap), 55, np.int8), np.full((H, cap), -66, np.int8)
    fp8.kv_cache_write_fp8(kc8, vc8, ke, ve, k, v, head_begin, off)
    return kc8, vc8, ke, ve


def test_write_places_rows_like_the_bf16_cache_write_and_leaves_the_rest_alone():
    rng = np.random.default_rng(4)
    n, Hs, d, H, cap, hb, off = 37, 5, 64, 3, 100, 1, 40
    k = wl.bf16_round(rng.standard_normal((n, Hs, d), dtype=np.float32))
    v = wl.bf16_round(rng.standard_normal((n, Hs, d), dtype=np.float32) * 7)
    kc8, vc8, ke, ve = quantise(k, v, H, cap, hb, off)
    touched = np.zeros(cap, bool)
    touched[off:off + n] = True
    assert np.all(kc8[:, ~touched] == 0xAB) and np.all(vc8[:, ~touched] == 0xCD)
    assert np.all(ke[:, ~touched] == 55) and np.all(ve[:, ~touched] == -66)
    # row (h, off + r) holds source row r of head hb + h: quantise that row alone and compare (numpy slicing)
    for h in range(H):
        for r in (0, 11, n - 1):
            x = v[r, hb + h]
            e = fp8.row_exponent(x)
            assert ve[h, off + r] == e
            assert np.array_equal(vc8[h, off + r], np.array([fp8.e4m3_encode(float(t) / 2.0 ** e) for t in x], np.uint8))


def test_round_trip_error_bound_and_exact_bf16_representability():
    rng = np.random.default_rng(5)
    n, H, d = 64, 2, 128
    k = wl.bf16_round(rng.standard_normal((n, H, d), dtype=np.float32) * np.float32(10.0) ** rng.uniform(-4, 3, (n, H, 1)).astype(np.float32))
    v = wl.bf16_round(rng.standard_normal((n, H, d), dtype=np.float32))
    v[5, 1] = 0.0                                          # an all-zero row
    kc8, vc8, ke, ve = quantise(k, v, H, n, 0, 0)
    for src, c8, ex in ((k, kc8, ke), (v, vc8, ve)):
        deq = fp8.kv_cache_dequant_fp8(c8, ex)            # [H, n, d]
        want = np.transpose(src, (1, 0, 2)).astype(np.float64)
        scale = 2.0 ** ex.astype(np.float64)[:, :, None]
        # half an ulp of a 4-significant-bit number (2^-4 relative), or half a subnormal step (2^-10 of the scale)
        assert np.all(np.abs(deq - want) <= np.maximum(np.abs(want) * 2.0 ** -4, scale * 2.0 ** -10) * (1 + 1e-12))
        assert np.array_equal(wl.bf16_round(deq), deq), "dequantised values must be exact BF16 numbers"
        assert np.all(np.abs(deq) <= np.abs(want).max(axis=2, keepdims=True) * (1 + 2.0 ** -4))
    assert np.all(vc8[1, 5] == 0) and ve[1, 5] == -100
    # a row of exactly representable values (4 significant bits, one binade range) survives unchanged
    x = np.array([[[1.0, -1.125, 0.4375, 448.0 / 256, 0.0, 2.0 ** -9, -0.15625, 0.875]]], np.float32)
    c8, _, ex, _ = quantise(x, x, 1, 1, 0, 0)
    assert np.array_equal(fp8.kv_cache_dequant_fp8(c8, ex)[0, 0], x[0, 0])
    # clamped scale: the row saturates instead of overflowing
    big = np.array([[[1e6, -3e5, 1.0, 0.0, 0.0, 0.0, 0.0, 0.0]]], np.float32)
    c8, _, ex, _ = quantise(big, big, 1, 1, 0, 0)
    assert ex[0, 0] == 7 and np.array_equal(fp8.kv_cache_dequant_fp8(c8, ex)[0, 0, :3], np.array([57344.0, -57344.0, 1.0], np.float32))


def test_bad_arguments_are_rejected():
    k = np.zeros((4, 2, 8), np.float32)
    c8, e = np.zeros((2, 8, 8), np.uint8), np.zeros((2, 8), np.int8)
    with pytest.raises(ValueError):
        fp8.kv_cache_write_fp8(c8, c8.copy(), e, e.copy(), k, k, 0, 5)      # 5 + 4 > capacity
    with pytest.raises(ValueError):
        fp8.kv_cache_write_fp8(c8, c8.copy(), e, e.copy(), k, k, 1, 0)      # head_begin + H > H_src
