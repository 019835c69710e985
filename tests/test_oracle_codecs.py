"""Pins for the oracle's element / scale codecs (not gpu).  Each test cites what fixes the value:
the paper (P:n = /root/reference/PAPER.md line n), a library (ml_dtypes) or exact rational
arithmetic."""
from fractions import Fraction

import ml_dtypes
import numpy as np

from oracle import sharq_oracle as so
from oracle import hif4_oracle as ho

F32 = np.float32


def all_bf16_as_f32():
    u = np.arange(65536, dtype=np.uint16)
    f = so.bf16_to_f32(u)
    return f[np.isfinite(f)]


def test_e2m1_decode_table_is_the_papers():
    assert so.e2m1_decode(np.arange(8, dtype=np.uint8)).tolist() == [0, .5, 1, 1.5, 2, 3, 4, 6]
    assert so.e2m1_decode(np.arange(8, 16, dtype=np.uint8)).tolist()[1:] == [-.5, -1, -1.5, -2, -3, -4, -6]


def test_e2m1_encode_matches_ml_dtypes_on_all_bf16_and_random_fp32():
    f = all_bf16_as_f32()
    rng = np.random.default_rng(0)
    r = np.concatenate([f, (rng.standard_normal(2_000_000) * 3).astype(F32),
                        rng.uniform(-7, 7, 2_000_000).astype(F32)])
    want = r.astype(ml_dtypes.float4_e2m1fn).view(np.uint8) & 0xF
    got = so.e2m1_encode(r)
    assert np.array_equal(got, want)


def test_e2m1_encode_is_nearest_with_ties_to_even_in_exact_arithmetic():
    grid = [Fraction(x) for x in (0, .5, 1, 1.5, 2, 3, 4, 6)]
    vals = [0.0, 0.1, 0.25, 0.2500001, 0.5, 0.74999, 0.75, 1.0, 1.25, 1.26, 1.75, 2.0, 2.5, 2.51, 3.5,
            4.9999, 5.0, 5.0001, 6.0, 7.0, 1e30]
    for v in vals:
        fv = Fraction(float(F32(v)))
        dist = [abs(fv - g) for g in grid]
        m = min(dist)
        cands = [i for i, d in enumerate(dist) if d == m]
        want = [c for c in cands if c % 2 == 0][0] if len(cands) > 1 else cands[0]
        assert so.e2m1_encode(np.array([v], F32))[0] == want, v
        assert so.e2m1_encode(np.array([-v], F32))[0] == want | 8, v
    assert so.e2m1_encode(np.array([-0.0], F32))[0] == 8         # sign kept on zero


def test_e4m3_closed_forms_from_the_paper():
    # P:390 bias 7; P:394 448*6 = 2688; P:483-484 max 2^11*1.3125, min 2^-10 (= 2^-9 * 0.5)
    assert so.e4m3_decode(np.array([0x7E], np.uint8))[0] == 448.0
    assert 448.0 * 6.0 == 2688.0 == 2.0 ** 11 * 1.3125
    assert so.e4m3_decode(np.array([0x01], np.uint8))[0] == 2.0 ** -9
    assert so.e4m3_decode(np.array([0x01], np.uint8))[0] * 0.5 == 2.0 ** -10
    assert so.e4m3_decode(np.array([0x38], np.uint8))[0] == 1.0   # exponent field 7 = bias


def test_e4m3_codec_matches_ml_dtypes():
    codes = np.arange(0x7F, dtype=np.uint8)
    assert np.array_equal(so.e4m3_decode(codes), codes.view(ml_dtypes.float8_e4m3fn).astype(F32))
    rng = np.random.default_rng(1)
    x = np.concatenate([np.exp(rng.uniform(np.log(2.0 ** -12), np.log(600.0), 3_000_000)).astype(F32),
                        so.e4m3_decode(codes), np.array([0, 2.0 ** -10, 2.0 ** -10 * 1.0001, 448, 464, 1e9], F32)])
    # exact midpoints between neighbouring codes
    d = so.e4m3_decode(codes).astype(np.float64)
    x = np.concatenate([x, ((d[:-1] + d[1:]) / 2).astype(F32)])
    want = np.minimum(x, F32(448)).astype(ml_dtypes.float8_e4m3fn).view(np.uint8)
    assert np.array_equal(so.e4m3_encode(x), want)


def test_e8m0_decode_matches_ml_dtypes_and_encode_is_smallest_power_of_two_not_below():
    codes = np.arange(255, dtype=np.uint8)
    assert np.array_equal(so.e8m0_decode(codes), codes.view(ml_dtypes.float8_e8m0fnu).astype(F32))
    rng = np.random.default_rng(2)
    x = np.exp(rng.uniform(np.log(1e-30), np.log(1e30), 20000)).astype(F32)
    x = np.concatenate([x, np.ldexp(F32(1), np.arange(-126, 127)).astype(F32),
                        np.nextafter(np.ldexp(F32(1), np.arange(-100, 100)).astype(F32), F32(np.inf))])
    got = so.e8m0_encode_rp(x).astype(int) - 127
    for xv, e in zip(x.tolist(), got.tolist()):
        fx = Fraction(xv)
        assert Fraction(2) ** e >= fx and Fraction(2) ** (e - 1) < fx, (xv, e)
    assert so.e8m0_encode_rp(np.array([0], F32))[0] == 0


def test_mxfp4_scale_cheap_form_equals_exact_definition():
    """R8: code = rp(RN(a*C6)) must be the smallest 2^e >= a/6 (exact rationals); checked around
    every binade edge 6*2^e and on random bf16 magnitudes."""
    rng = np.random.default_rng(3)
    a = np.concatenate([
        so.bf16_to_f32(rng.integers(0x0800, 0x7F00, 50000).astype(np.uint16)),
        np.concatenate([np.nextafter(F32(6) * np.ldexp(F32(1), np.arange(-60, 60)).astype(F32), F32(s))
                        for s in (np.inf, -np.inf)]),
        F32(6) * np.ldexp(F32(1), np.arange(-60, 60)).astype(F32)])
    code = so.e8m0_encode_rp(a.astype(F32) * so.C6).astype(int) - 127
    for av, e in zip(a.tolist(), code.tolist()):
        t = Fraction(av) / 6
        assert Fraction(2) ** e >= t and Fraction(2) ** (e - 1) < t, (av, e)


def test_c6_is_rn_of_one_sixth():
    assert Fraction(float(so.C6)) == min((Fraction(float(c)) for c in
                                          (np.nextafter(so.C6, F32(0)), so.C6, np.nextafter(so.C6, F32(1)))),
                                         key=lambda c: abs(c - Fraction(1, 6)))


# ---------------------------------------------------------------- HiF4
def test_hif4_closed_forms_from_the_paper():
    # Table 7
    assert ho.e6m2_decode(np.array([0xFE], np.uint8))[0] == 2.0 ** 15 * 1.5
    assert ho.e6m2_decode(np.array([0x00], np.uint8))[0] == 2.0 ** -48
    assert ho.s1p2_decode(np.array([7, 15, 1, 9, 0], np.uint8)).tolist() == [1.75, -1.75, .25, -.25, 0]
    # unit = 64*4 + 32 = 288 bits = 4.5 bits/value
    assert 64 * 4 + 32 == 288 and 288 / 64 == 4.5
    # in-unit max 2^(1+1)*1.75 = 7, min 0.25; global max 2^18*1.3125, min 2^-50 (Table 8)
    top = np.array([0xFE | 0xFF << 8 | 0xFFFF << 16], np.uint32)
    v = ho.hif4_decode_units(np.full((1, 64), 7, np.uint8), top)
    assert v.max() == 2.0 ** 15 * 1.5 * 4 * 1.75 == 2.0 ** 18 * 1.3125       # E6M2max * 7 (Table 8)
    one = np.array([0xC0 | 0xFF << 8 | 0xFFFF << 16], np.uint32)             # E6M2 = 1.0
    assert ho.hif4_decode_units(np.full((1, 64), 7, np.uint8), one).max() == 7.0
    lo = np.array([0x00], np.uint32)
    assert ho.hif4_decode_units(np.full((1, 64), 1, np.uint8), lo).min() == 2.0 ** -50


def test_hif4_reciprocal_table_is_bf16_of_exact_reciprocal():
    for m in range(4):
        exact = Fraction(4, 4 + m)
        got = Fraction(float(ho.REC_LUT[m]))
        # nearest bf16 (8 significant bits) to 1/1.M
        cands = [Fraction(n, 256) for n in range(128, 257)]
        assert got == min(cands, key=lambda c: abs(c - exact))
    assert Fraction(float(ho.ONE_SEVENTH_BF16)) == min((Fraction(n, 1024) for n in range(128, 256)),
                                                       key=lambda c: abs(c - Fraction(1, 7)))


def test_hif4_alg1_derived_vectors():
    """Hand-derived from Algorithm 1 under R9-R11: 64 x 7.0 and 64 x 1.0."""
    bf = lambda v: so.f32_to_bf16(np.full((1, 64), v, F32))
    c, m = ho.hif4_encode_units(bf(7.0))
    # SF = bf16(7 * 0.142578125 = 0.998046875) = 1.0 -> E6M2 0xC0; 7*1 >= 4 and 3.5 >= 2 -> E1 = 1
    assert m[0] == (0xC0 | 0xFF << 8 | 0xFFFF << 16) and (c == 7).all()
    assert (ho.hif4_decode_units(c, m) == 7.0).all()
    c, m = ho.hif4_encode_units(bf(1.0))
    # SF = 0.142578125 = 1.140625 * 2^-3 -> 1.M rounds to 1.25 -> E6M2 = (45 << 2) | 1 = 0xB5
    # REC = 0.80078125 * 8 = 6.40625 >= 4 -> E1_8 = 1; 3.203125 >= 2 -> E1_16 = 1; 1.6015625 -> 1.5
    assert m[0] == (0xB5 | 0xFF << 8 | 0xFFFF << 16) and (c == 6).all()
    assert (ho.hif4_decode_units(c, m) == 0.9375).all()


def test_hif4_round_trip_on_grid_and_threshold_predicates():
    rng = np.random.default_rng(5)
    # random units ON the HiF4 grid whose maximum pins the scale: one element = 7 * base
    for base_code in (0xC0, 0xB5, 0x90, 0xE2):
        base = float(ho.e6m2_decode(np.array([base_code], np.uint8))[0])
        codes = rng.integers(0, 16, (200, 64)).astype(np.uint8)
        meta = (np.uint32(base_code) | (rng.integers(0, 256, 200).astype(np.uint32) << 8)
                | (rng.integers(0, 65536, 200).astype(np.uint32) << 16))
        vals = ho.hif4_decode_units(codes, meta)
        assert np.array_equal(so.bf16_to_f32(so.f32_to_bf16(vals)), vals)    # grid values are bf16-exact
    x = (rng.standard_normal((500, 64)) * np.exp(rng.uniform(-3, 3, (500, 1)))).astype(F32)
    xb = so.f32_to_bf16(x)
    c, m = ho.hif4_encode_units(xb)
    rec = ho.e6m2_reciprocal((m & 0xFF).astype(np.uint8)).astype(np.float64)
    A = np.abs(so.bf16_to_f32(xb)).astype(np.float64)
    V16 = A.reshape(-1, 16, 4).max(-1); V8 = V16.reshape(-1, 8, 2).max(-1)
    e8 = ((m[:, None] >> (8 + np.arange(8))) & 1).astype(bool)
    e16 = ((m[:, None] >> (16 + np.arange(16))) & 1).astype(bool)
    assert np.array_equal(e8, V8 * rec[:, None] >= 4)
    assert np.array_equal(e16, V16 * rec[:, None] * np.where(np.repeat(e8, 2, 1), .5, 1) >= 2)
    # reconstruction error of every element is at most half a S1P2 step at its scale (+ bf16 rounding)
    d = ho.hif4_decode_units(c, m).astype(np.float64)
    step = ho.e6m2_decode((m & 0xFF).astype(np.uint8)).astype(np.float64)[:, None] * 0.25 \
        * np.where(np.repeat(e8, 8, 1), 2, 1) * np.where(np.repeat(e16, 4, 1), 2, 1)
    sat = (c & 7) == 7
    X = so.bf16_to_f32(xb).astype(np.float64)
    assert (np.abs(X - d)[~sat] <= step[~sat] * (0.5 + 2.0 ** -6) * 1.3).all()


def test_hif4_significands_and_the_fp8_question():
    """SURVEY.md 8(f) N4 (the FP8-rate HiF4 study), the arithmetic behind DESIGN.md's conclusion.  Every HiF4 value is
    +-(4 + m) * k * 2^p (E6M2 mantissa 1.m, S1P2 magnitude k / 4, the E1 shifts and the exponent in p; Eq. 15 P:467,
    Table 7): its significand (4 + m) * k <= 49 needs at most 6 bits, so bf16 (8 bits) holds every value
    exactly -- what the B200 path relies on -- while FP8 does not: e4m3 (4 bits) represents only 21 of the 28 nonzero
    (m, k) combinations, e5m2 (3 bits) 16.  An exact FP8 path therefore needs a two-term split of BOTH operands (four
    FP8 GEMMs at twice the bf16 rate = twice the bf16 time); the per-unit mantissa cannot go into a block scale either,
    because tcgen05's FP8 block scales are powers of two (UE8M0)."""
    def sig_bits(n):
        while n % 2 == 0:
            n //= 2
        return n.bit_length()
    pairs = [(m, k) for m in range(4) for k in range(1, 8)]
    need = [sig_bits((4 + m) * k) for m, k in pairs]
    assert max(need) == 6 and max((4 + m) * k for m, k in pairs) == 49
    assert sum(b <= 4 for b in need) == 21 and sum(b <= 3 for b in need) == 16 and sum(b <= 8 for b in need) == 28
    # the oracle's decode agrees: every decoded value of random units has an odd part below 2^6, and e4m3 misses some
    rng = np.random.default_rng(3)
    codes = rng.integers(0, 16, (64, 64)).astype(np.uint8)
    meta = (rng.integers(0x80, 0xF0, 64).astype(np.uint32) | (rng.integers(0, 1 << 24, 64).astype(np.uint32) << 8))
    v = np.abs(ho.hif4_decode_units(codes, meta).astype(np.float64)).ravel()
    v = v[v > 0]
    mant, _ = np.frexp(v)
    sig = (mant * 2.0 ** 6)
    assert (sig == np.round(sig)).all()                                   # 6 bits suffice
    exact_e4m3 = np.array(v, np.float32).astype(ml_dtypes.float8_e4m3fn).astype(np.float64) == v
    in_range = (v <= 448) & (v >= 2.0 ** -6)
    assert 0.5 < exact_e4m3[in_range].mean() < 0.95                       # ... and four bits do not
