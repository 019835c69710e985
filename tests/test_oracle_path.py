"""Pins for the oracle's path (norm -> mask -> backbone -> residual -> GEMMs); not gpu.
P:n = /root/reference/PAPER.md line n."""
import itertools
import math
from fractions import Fraction

import ml_dtypes
import numpy as np
import pytest

import sharq_inputs as si
from oracle import sharq_oracle as so

F32 = np.float32


@pytest.fixture(scope="module")
def small():
    T, K, D = 8, 1024, 256
    x = si.activations(T, K, config=1)
    g = si.gamma(K)
    w = si.weight(D, K)
    return x, g, w


# ------------------------------------------------------------------ O1 norm
def test_canonical_sum_against_fsum_and_special_cases():
    rng = np.random.default_rng(0)
    for K in (256, 768, 1024, 3584, 4096):
        x = rng.standard_normal((3, K)).astype(F32)
        s = so.canonical_sum(x, squares=True)
        for t in range(3):
            exact = math.fsum((float(v) ** 2 for v in x[t]))
            assert abs(float(s[t]) - exact) <= K * 2.0 ** -24 * exact
        # powers of two sum exactly whatever the order
        p = np.ldexp(F32(1), rng.integers(-3, 4, (2, K))).astype(F32)
        assert np.array_equal(so.canonical_sum(p, squares=False), p.astype(np.float64).sum(1).astype(F32))
    # order pin: a permutation inside one 8-leaf that changes a naive left-to-right sum
    x = np.zeros((1, 1024), F32); x[0, 0] = 2.0 ** 24; x[0, 1] = 1.0; x[0, 2] = 1.0
    assert so.canonical_sum(x, False)[0] == 2.0 ** 24            # (2^24+1)+1 = 2^24 in fp32
    x[0, 0], x[0, 2] = 1.0, 2.0 ** 24
    assert so.canonical_sum(x, False)[0] == 2.0 ** 24 + 2        # (1+1)+2^24


def test_rmsnorm_against_fp64_and_exact_case():
    x = si.activations(4, 4096, config=1); g = si.gamma(4096)
    X = so.bf16_to_f32(so.normalize(x, so.NORM_RMS, g)).astype(np.float64)
    xf = so.bf16_to_f32(x).astype(np.float64); gf = so.bf16_to_f32(g).astype(np.float64)
    ref = xf / np.sqrt((xf ** 2).mean(1, keepdims=True) + 1e-6) * gf
    assert np.abs(X - ref).max() <= np.abs(ref).max() * 2.0 ** -7          # two bf16 roundings
    assert (np.abs(X - ref) <= np.abs(ref) * (2.0 ** -8 + 2.0 ** -8 + 2.0 ** -15) + 1e-30).all()
    # exact case: x = +-2 everywhere, gamma = 1, eps = 0 -> X = +-1 exactly
    s = np.where(np.arange(512) % 3 == 0, -2.0, 2.0).astype(F32)[None, :]
    X = so.normalize(so.f32_to_bf16(s), so.NORM_RMS, so.f32_to_bf16(np.ones(512, F32)), eps=0.0)
    assert np.array_equal(so.bf16_to_f32(X), s / 2)
    # layernorm: mean 0 / unit variance up to bf16
    xl = so.f32_to_bf16((np.random.default_rng(1).standard_normal((2, 1024)) * 3 + 5).astype(F32))
    X = so.bf16_to_f32(so.normalize(xl, so.NORM_LAYER, so.f32_to_bf16(np.ones(1024, F32)),
                                    so.f32_to_bf16(np.zeros(1024, F32)))).astype(np.float64)
    assert abs(X.mean()) < 1e-2 and abs(X.std() - 1) < 1e-2


# ------------------------------------------------------------------ O3 masks
def _best_mask_bruteforce(scores):
    """Among the 6 two-of-four masks: lexicographically largest sorted kept scores, then lowest indices."""
    best = None
    for c in itertools.combinations(range(4), 2):
        key = (tuple(sorted((scores[i] for i in c), reverse=True)), tuple(-i for i in c))
        if best is None or key > best[0]:
            best = (key, c)
    return best[1]


def test_pair_mask_exhaustive_small_alphabet():
    """Every chunk of 8 with values in {0,+-1,+-2,+-3} restricted to score patterns: all 4^4 score
    tuples over 4 distinct magnitudes x all placements of the max inside the pair (every tie pattern)."""
    vals = so.f32_to_bf16(np.array([0, 1, 2, 3], F32))
    rows = []
    for sc in itertools.product(range(4), repeat=4):
        for lay in range(16):                      # which element of each pair carries the score
            ch = []
            for p in range(4):
                hi, lo = vals[sc[p]], vals[0] if sc[p] == 0 else vals[sc[p] - 1]
                sign = 0x8000 if (lay >> p) & 1 else 0
                ch += ([hi | sign, lo] if (lay >> p) & 1 else [lo, hi | sign])
            rows.append(ch)
    X = np.array(rows, dtype=np.uint16).reshape(1, -1)
    keep, nib = so.mask_pair48(X)
    keep = keep.reshape(-1, 4, 2); nib = nib.reshape(-1)
    u = (X.reshape(-1, 4, 2) & 0x7FFF).max(-1)
    for n in range(u.shape[0]):
        c = _best_mask_bruteforce(u[n].tolist())
        assert nib[n] == c[0] | (c[1] << 2)
        assert keep[n].all(1).tolist() == [i in c for i in range(4)]
        assert (keep[n, :, 0] == keep[n, :, 1]).all()


def test_masks_on_random_data_and_24_exhaustive():
    x = si.activations(16, 1024, config=1)
    keep, nib = so.mask_pair48(x)
    assert (keep.reshape(16, -1, 8).sum(-1) == 4).all()                    # exactly N survivors per M
    assert ((nib & 3) < (nib >> 2)).all()                                  # ascending indices
    # the largest element of every chunk is in the backbone
    a = (x & 0x7FFF).reshape(16, -1, 8)
    assert np.take_along_axis(keep.reshape(16, -1, 8), a.argmax(-1)[..., None], -1).all()
    k24, n24 = so.mask_24(x)
    assert (k24.reshape(16, -1, 4).sum(-1) == 2).all()
    vals = so.f32_to_bf16(np.array([0, -1, 1, 2, -3], F32))
    allq = np.array(list(itertools.product(vals.tolist(), repeat=4)), dtype=np.uint16).reshape(1, -1)
    k, n = so.mask_24(allq)
    u = (allq.reshape(-1, 4) & 0x7FFF)
    for i in range(u.shape[0]):
        c = _best_mask_bruteforce(u[i].tolist())
        assert n[0, i] == c[0] | (c[1] << 2) and k.reshape(-1, 4)[i].tolist() == [j in c for j in range(4)]


# ------------------------------------------------------------------ O2/O4-O6 scales, residual
@pytest.mark.parametrize("fmt", [so.NVFP4, so.MXFP4])
def test_prepare_invariants(small, fmt):
    x, g, _ = small
    p = so.prepare(x, fmt=fmt, gamma_u16=g)
    T, K = x.shape
    Xf = so.bf16_to_f32(p["X"]).astype(np.float64)
    ts = p["ts"].astype(np.float64)
    if fmt == so.NVFP4:
        assert np.array_equal(p["ts"], (np.abs(Xf).max(1) / 2688.0).astype(F32))
    # scale = amax/6 (/ts) rounded to the scale format, evaluated in fp64 (BASELINE.json invariant)
    a_sp = np.where(p["keep"], np.abs(Xf), 0).reshape(T, -1, 32).max(-1)
    if fmt == so.NVFP4:
        want = np.minimum(a_sp / 6 / ts[:, None], 448).astype(F32).astype(ml_dtypes.float8_e4m3fn).view(np.uint8)
        assert (p["sp_sf"] == want).mean() > 0.999          # fp32 chain vs fp64: only boundary cases differ
        assert (np.abs(p["sp_sf"].astype(int) - want.astype(int)) <= 1).all()
        sf = so.e4m3_decode(p["sp_sf"]).astype(np.float64) * ts[:, None]
        assert (sf * 6 >= a_sp * (1 - 2.0 ** -4) - 1e-30).all()
    else:
        sf = so.e8m0_decode(p["sp_sf"]).astype(np.float64)
        assert (sf * 6 >= a_sp).all() and (sf * 3 < a_sp)[a_sp > 0].all()               # smallest 2^e >= a/6
    # every code on the grid; residual identity Eq. 8 exact in fp64
    assert (so.unpack_codes(p["sp_codes"]) < 16).all() and (so.unpack_codes(p["dn_codes"]) < 16).all()
    assert np.array_equal(p["R"].astype(np.float64) + p["Xsp_tilde"].astype(np.float64), Xf)
    assert np.array_equal(p["R"][~p["keep"]], so.bf16_to_f32(p["X"])[~p["keep"]])
    # Xsp_tilde equals what the stored bytes decode to (compression + metadata round trip)
    back = so.dequant_backbone(p)
    assert np.allclose(back, p["Xsp_tilde"], rtol=2 ** -22, atol=0)
    codes, keep2 = so.expand_backbone(p)
    assert np.array_equal(keep2, p["keep"])
    # Eq. 12: X - (Xsp~ + R~) == R - R~, and the element error bound of the residual quantizer
    Rt = so.dequant_residual(p)
    lhs = Xf - (p["Xsp_tilde"].astype(np.float64) + Rt)
    rhs = p["R"].astype(np.float64) - Rt
    assert np.abs(lhs - rhs).max() <= 2.0 ** -40 * np.abs(Xf).max()
    Gd = p["Gd"]
    sfd = (so.sf_decode(p["dn_sf"], fmt).astype(np.float64) * ts[:, None]).repeat(Gd, 1)
    dn = so.unpack_codes(p["dn_codes"]) & 7
    half_gap = np.array([.25, .25, .25, .25, .5, .5, 1.0, 1.0])[dn]                    # half the e2m1 gap at that code
    assert (np.abs(rhs)[dn < 7] <= (sfd * half_gap)[dn < 7] * (1 + 1e-6)).all()
    # outliers isolated: residual block scales are not larger than a plain dense quantizer's
    p0 = so.prepare(x, fmt=fmt, gamma_u16=g, _force_no_survivors=True)
    assert so.sf_decode(p["dn_sf"], fmt).astype(np.float64).sum() < so.sf_decode(p0["dn_sf"], fmt).astype(np.float64).sum()


def test_dense_only_special_case_equals_independent_nvfp4_quantizer(small):
    """Empty mask => R = X and the residual path is a plain NVFP4 quantizer: compare with an
    independent numpy + ml_dtypes implementation (casts done by the library)."""
    x, g, _ = small
    p = so.prepare(x, gamma_u16=g, _force_no_survivors=True)
    Xf = so.bf16_to_f32(p["X"])
    assert np.array_equal(p["R"], Xf)
    T, K = Xf.shape
    ts = (np.abs(Xf).max(1) / F32(2688)).astype(F32)
    amax = np.abs(Xf).reshape(T, K // 16, 16).max(-1)
    c6 = np.array([0x3E2AAAAB], np.uint32).view(F32)[0]
    sf8 = ((amax * c6) * (F32(1) / ts)[:, None]).astype(F32).astype(ml_dtypes.float8_e4m3fn)
    assert np.array_equal(sf8.view(np.uint8), p["dn_sf"])
    s_eff = sf8.astype(F32) * ts[:, None]
    q = (Xf * np.repeat(F32(1) / s_eff, 16, 1)).astype(F32).astype(ml_dtypes.float4_e2m1fn).view(np.uint8) & 0xF
    assert np.array_equal(q[:, 0::2] | (q[:, 1::2] << 4), p["dn_codes"])


def test_static_tensor_scale_and_zero_rows():
    x = si.activations(4, 512, config=1)
    x[1] = 0
    p = so.prepare(x, norm=so.NORM_NONE)
    assert p["ts"][1] == 1.0 and (p["sp_sf"][1] == 0).all() and (p["dn_codes"][1] == 0).all()
    ps = so.prepare(x, norm=so.NORM_NONE, x_tensor_scale=0.03125)
    assert (ps["ts"] == F32(0.03125)).all()


# ------------------------------------------------------------------ O8 weights, O7 linear
@pytest.mark.parametrize("fmt", [so.NVFP4, so.MXFP4, so.HIF4])
def test_weight_views_share_one_payload(small, fmt):
    _, _, w = small
    wq = so.quantize_weight(w, fmt)
    if fmt == so.NVFP4:
        assert np.array_equal(wq["sf_dn"][:, 0::2], wq["sf_sp"]) and np.array_equal(wq["sf_dn"][:, 1::2], wq["sf_sp"])
    assert np.array_equal(so.dequant_weight(wq, "sparse"), so.dequant_weight(wq, "dense"))
    Wf = so.bf16_to_f32(w).astype(np.float64)
    err = np.linalg.norm(so.dequant_weight(wq) - Wf) / np.linalg.norm(Wf)
    assert err < 0.13


@pytest.mark.parametrize("fmt", [so.NVFP4, so.MXFP4, so.HIF4])
def test_linear_against_blas_loops_and_eq13(small, fmt):
    x, g, w = small
    p = so.prepare(x, fmt=fmt, gamma_u16=g)
    wq = so.quantize_weight(w, fmt)
    Y = so.linear(p, wq)
    A = so.dequant_backbone(p) + so.dequant_residual(p)                 # Xsp~ + R~
    Wd = so.dequant_weight(wq)
    assert np.allclose(Y, A @ Wd.T, rtol=1e-11, atol=1e-11 * np.abs(Y).max())
    for (t, d) in ((0, 0), (3, 17), (7, 255)):
        assert math.isclose(so.linear_loops(p, wq, t, d), Y[t, d], rel_tol=1e-11, abs_tol=1e-12)
    sub = so.linear(p, wq, rows=np.array([1, 5]), cols=np.array([2, 200]))
    assert np.array_equal(sub, Y[np.ix_([1, 5], [2, 200])])
    # Eq. 13
    Xf = so.bf16_to_f32(p["X"]).astype(np.float64)
    Rt = so.dequant_residual(p)
    lhs = np.linalg.norm(Xf @ Wd.T - A @ Wd.T)
    rhs = np.linalg.norm(p["R"].astype(np.float64) - Rt) * np.linalg.svd(Wd, compute_uv=False)[0]
    assert lhs <= rhs * (1 + 1e-9)


def test_qualitative_ordering_of_path_combinations():
    """P:265, P:288 (Table 5): sparse-only >> plain dense NVFP4 >~ SharQ in activation error."""
    x = si.activations(32, 4096, config=1); g = si.gamma(4096)
    p = so.prepare(x, gamma_u16=g)
    p0 = so.prepare(x, gamma_u16=g, _force_no_survivors=True)
    Xf = so.bf16_to_f32(p["X"]).astype(np.float64)
    n = np.linalg.norm
    e_sparse = n(so.dequant_backbone(p) - Xf) / n(Xf)
    e_dense = n(so.dequant_residual(p0) - Xf) / n(Xf)
    e_sharq = n(so.dequant_backbone(p) + so.dequant_residual(p) - Xf) / n(Xf)
    assert e_sparse > 2 * e_dense and e_dense > 2 * e_sharq


def _nearest_bf16_exact(v: Fraction) -> int:
    """Nearest bf16 bit pattern of an exact rational (ties to even), by brute force over the two neighbours."""
    if v == 0:
        return 0
    sign = 0x8000 if v < 0 else 0
    a = abs(v)
    e = math.floor(math.log2(float(a))) if a >= Fraction(1, 2 ** 120) else -126
    while Fraction(2) ** e > a:
        e -= 1
    while Fraction(2) ** (e + 1) <= a:
        e += 1
    e = max(e, -126)                                   # subnormals share the spacing of the lowest binade
    ulp = Fraction(2) ** (e - 7)
    q, r = divmod(a, ulp)
    q = int(q)
    if r * 2 > ulp or (r * 2 == ulp and (q & 1)):
        q += 1
    val = q * ulp
    bits = int(np.float32(float(val)).view(np.uint32)) >> 16      # val is a bf16 value: exact in fp32
    return sign | bits


def test_residual_add_is_one_rounding_of_the_exact_sum():
    """sharq_prepare_add's h = bf16(x + r): the oracle's fp32 add + RNE equals the exactly
    rounded rational sum, on random pairs and on pairs built to stress the double rounding (exponent gaps of
    8..24 around tie points) and cancellation."""
    rng = np.random.default_rng(26587)
    a = si.to_bf16_bits((rng.standard_normal(3000) * 10.0 ** rng.integers(-6, 6, 3000)).astype(np.float32))
    b = si.to_bf16_bits((rng.standard_normal(3000) * 10.0 ** rng.integers(-6, 6, 3000)).astype(np.float32))
    # adversarial: big = 1.xxxxxxx * 2^0, small = +-(2^-8 +- 2^-k), +-2^-9 ..., and near cancellation
    big = (0x3F80 + rng.integers(0, 128, 600)).astype(np.uint16)
    gaps = rng.integers(8, 26, 600)
    small_f = np.ldexp(1.0, -gaps) * rng.choice([1.0, -1.0, 1.5, -1.5, 1.0078125, 0.9921875], 600)
    small = si.to_bf16_bits(small_f.astype(np.float32))
    a = np.concatenate([a, big, big, np.array([0x0001, 0x8001, 0x0080, 0x7F7F], np.uint16)])
    b = np.concatenate([b, small, (big ^ 0x8000) + rng.integers(0, 3, 600).astype(np.uint16),
                        np.array([0x0001, 0x0001, 0x8001, 0x0000], np.uint16)])
    got = so.residual_add(a, b)
    fa, fb = si.bf16_bits_to_f32(a), si.bf16_bits_to_f32(b)
    for i in range(a.size):
        exact = Fraction(float(fa[i])) + Fraction(float(fb[i]))
        want = _nearest_bf16_exact(exact)
        if exact == 0:                                 # x + (-x) = +0 under round-to-nearest
            want = 0x8000 if (a[i] & 0x8000 and b[i] & 0x8000) else 0
        assert int(got[i]) == want, (hex(a[i]), hex(b[i]), hex(got[i]), hex(want))


# ------------------------------------------------------------------ O1 LayerNorm branch (R3)
def _rne_bf16_fraction(v: Fraction) -> Fraction:
    """Nearest bf16 value (8 significant bits, ties to the even significand) of an exact rational, by search."""
    if v == 0:
        return Fraction(0)
    s, a = (-1 if v < 0 else 1), abs(v)
    e = 0
    while Fraction(2) ** (e + 1) <= a:
        e += 1
    while Fraction(2) ** e > a:
        e -= 1
    q = Fraction(2) ** (e - 7)                       # spacing of the bf16 grid in [2^e, 2^(e+1))
    n = a / q
    lo = n.numerator // n.denominator
    r = n - lo
    if r > Fraction(1, 2) or (r == Fraction(1, 2) and lo % 2 == 1):
        lo += 1
    return s * lo * q


def _layernorm_fp64(x_u16, g_u16, b_u16, eps, variant="paper"):
    """fp64 ((x - mu) / sqrt(var + eps)) * gamma + beta (P:155 'LayerNorm'), and the plausible mistakes the pin
    must reject: beta sign flipped, beta added before gamma, unbiased (N - 1) variance."""
    xf = so.bf16_to_f32(x_u16).astype(np.float64)
    g = so.bf16_to_f32(g_u16).astype(np.float64)
    b = so.bf16_to_f32(b_u16).astype(np.float64)
    mu = xf.mean(1, keepdims=True)
    N = xf.shape[1]
    var = ((xf - mu) ** 2).sum(1, keepdims=True) / (N - 1 if variant == "nm1" else N)
    n = (xf - mu) / np.sqrt(var + eps)
    if variant == "beta_sign":
        return n * g - b, n * g
    if variant == "beta_first":
        return (n + b) * g, n * g
    return n * g + b, n * g


@pytest.mark.parametrize("K", [16, 256, 1024])
def test_layernorm_against_fp64_with_affine_and_mutations(K):
    """gamma != 1, beta != 0: the oracle's LayerNorm branch stays inside the three-bf16-rounding error bound of the
    fp64 definition on EVERY element, and each plausible mistake (beta sign, beta before gamma, N - 1 variance, at
    K = 16 where it moves every element by 3 %) violates the same bound on the same data, so the pin does discriminate."""
    rng = np.random.default_rng(K)
    x = so.f32_to_bf16((rng.standard_normal((6, K)) * 3 + 5).astype(F32))
    g = so.f32_to_bf16((rng.random(K) + 0.5).astype(F32))
    b = so.f32_to_bf16(rng.standard_normal(K).astype(F32))
    eps = 1e-6
    X = so.bf16_to_f32(so.normalize(x, so.NORM_LAYER, g, b, eps)).astype(np.float64)

    def within(ref, ng):
        # h = bf16(c*rstd), v = bf16(h*gamma): 2 x 2^-8 relative on |n*gamma| (+ fp32 slack); final bf16(v + beta):
        # 2^-8 relative on the result
        bound = np.abs(ng) * (2.0 ** -7 + 2.0 ** -14) + (np.abs(ref) + np.abs(ng) * 2.0 ** -7) * 2.0 ** -8 + 1e-30
        return np.abs(X - ref) <= bound

    ref, ng = _layernorm_fp64(x, g, b, eps)
    assert within(ref, ng).all()
    for variant in ("beta_sign", "beta_first") + (("nm1",) if K == 16 else ()):
        bad, ng_bad = _layernorm_fp64(x, g, b, eps, variant)
        assert (~within(bad, ng_bad)).mean() > 0.25, variant          # a large share of elements must fail


def test_layernorm_exact_power_of_two_case():
    """x = +-2^j balanced -> mu = 0, var = 4^j, rstd = 2^-j exactly (eps = 0); gamma = 2^a, beta = 2^b:
    X = +-2^a + 2^b, exactly representable in bf16 for |a - b| <= 6.  By hand, no arithmetic of the oracle."""
    K = 512
    for j, a, bexp in ((3, 1, -2), (-4, -1, 2), (0, 0, 0), (5, 3, -3)):
        sgn = np.where(np.arange(K) % 2 == 0, 1.0, -1.0)
        x = so.f32_to_bf16((sgn * 2.0 ** j).astype(F32))[None, :]
        g = so.f32_to_bf16(np.full(K, 2.0 ** a, F32))
        b = so.f32_to_bf16(np.full(K, 2.0 ** bexp, F32))
        X = so.bf16_to_f32(so.normalize(x, so.NORM_LAYER, g, b, eps=0.0))[0]
        assert np.array_equal(X, (sgn * 2.0 ** a + 2.0 ** bexp).astype(F32)), (j, a, bexp)
    # beta sign and gamma/beta order on an asymmetric hand case: x = {+2^j, -2^j}, gamma = 4, beta = -0.5 -> {3.5, -4.5}
    x = so.f32_to_bf16(np.array([[8.0, -8.0] * 128], F32))
    X = so.bf16_to_f32(so.normalize(x, so.NORM_LAYER, so.f32_to_bf16(np.full(256, 4.0, F32)),
                                    so.f32_to_bf16(np.full(256, -0.5, F32)), eps=0.0))[0]
    assert np.array_equal(X, np.array([3.5, -4.5] * 128, F32))


def test_layernorm_rounding_points_in_exact_rationals():
    """DESIGN.md R3's rounding points, X = bf16(bf16(bf16(c * rstd) * gamma) + beta) with c = x - mu in fp32, on a
    hand-made row where each of the bf16 roundings changes the answer in some columns: x in {+-1, +-7} balanced -> mu = 0,
    var = 25, rstd = RN(1 / 5) in fp32.  Expected values computed in exact rational arithmetic with a brute-force
    nearest-bf16 search; the variants that skip a rounding are shown to differ, so the pin is sensitive to them."""
    K = 256
    vals = np.array([1.0, -1.0, 7.0, -7.0] * (K // 4), F32)
    x = so.f32_to_bf16(vals)[None, :]
    rng = np.random.default_rng(7)
    g = so.f32_to_bf16((rng.random(K) + 0.5).astype(F32))       # per-column gamma / beta: bf16 values, exact rationals
    b = so.f32_to_bf16((rng.standard_normal(K) * 0.1).astype(F32))
    X = so.bf16_to_f32(so.normalize(x, so.NORM_LAYER, g, b, eps=0.0))[0]
    rstd = F32(1.0) / F32(5.0)                                   # sqrt(25) = 5 exactly; the one fp32 value RN(1/5)
    skipped = {"h": 0, "v": 0}
    for i, xv in enumerate(vals.tolist()):
        gq, bq = Fraction(float(so.bf16_to_f32(g[i:i + 1])[0])), Fraction(float(so.bf16_to_f32(b[i:i + 1])[0]))
        n32 = Fraction(float(F32(xv) * rstd))                    # fp32 product c * rstd (one RN)
        h = _rne_bf16_fraction(n32)
        v = _rne_bf16_fraction(h * gq)
        want = _rne_bf16_fraction(v + bq)
        assert Fraction(float(X[i])) == want, (i, xv)
        skipped["h"] += _rne_bf16_fraction(_rne_bf16_fraction(n32 * gq) + bq) != want
        skipped["v"] += _rne_bf16_fraction(h * gq + bq) != want
    assert skipped["h"] > 10 and skipped["v"] > 10, skipped


def test_hif4_residual_is_x_minus_decoded_backbone():
    """Eq. 8 on the HiF4 path, directly: R + D_sp(Q_sp(M (.) X)) == X exactly in fp64 wherever the
    subtraction was exact, dropped positions carry X bit for bit, and the stored backbone decodes (Eq. 15,
    P:467) to the same values the residual was formed against."""
    x = si.activations(6, 1024, config=4)
    p = so.prepare(x, fmt=so.HIF4, mask=so.MASK_24, norm=so.NORM_NONE)
    Xf = so.bf16_to_f32(p["X"]).astype(np.float64)
    d = so.dequant_backbone(p)                                     # rebuilt from sp_codes / sp_meta / sp_sf only
    assert np.array_equal(d, p["Xsp_tilde"].astype(np.float64))
    assert np.array_equal(p["R"][~p["keep"]].view(np.uint32), so.bf16_to_f32(p["X"])[~p["keep"]].view(np.uint32))
    assert (p["keep"].reshape(6, -1, 4).sum(-1) == 2).all()
    exact = p["R"].astype(np.float64) + d == Xf
    assert exact.mean() > 0.999                                    # fp32 subtraction of nearby values: Sterbenz
    assert np.abs(p["R"].astype(np.float64) + d - Xf).max() <= np.abs(Xf).max() * 2.0 ** -24


# ------------------------------------------------------------------ Table 5 path combinations
@pytest.mark.parametrize("fmt", [so.NVFP4, so.MXFP4])
def test_dense_dense_paths(fmt):
    """Dense+Dense: the first path is a plain dense quantiser of X -- byte for byte the 'dense-only special case' of
    prepare() (itself pinned against ml_dtypes) -- and the second path is the same quantiser applied to the exact
    residual; the two-path error is far below the one-path error (6.63 vs the NVFP4 baseline's 6.95)."""
    x = si.activations(8, 1024, config=1); g = si.gamma(1024)
    pp = so.prepare_paths(x, so.PATH_DENSE_DENSE, fmt=fmt, gamma_u16=g)
    p0 = so.prepare(x, fmt=fmt, gamma_u16=g, _force_no_survivors=True)
    assert np.array_equal(pp["a0_codes"], p0["dn_codes"]) and np.array_equal(pp["a0_sf"], p0["dn_sf"])
    Xf = so.bf16_to_f32(pp["X"]).astype(np.float64)
    assert np.array_equal(pp["R"].astype(np.float64) + pp["A0"].astype(np.float64), Xf)          # Eq. 8, exact
    # second path = the dense quantiser on R: re-run it through prepare()'s own dense branch on a bf16-free route
    Gd = 16 if fmt == so.NVFP4 else 32
    ts = pp["ts"]; inv_ts = (F32(1) / ts).astype(F32)
    a = np.abs(pp["R"]).reshape(8, -1, Gd).max(-1)
    sf, s_eff, inv = so._block_scale(a, fmt, ts, inv_ts)
    assert np.array_equal(sf, pp["a1_sf"])
    assert (so.sf_decode(pp["a1_sf"], fmt).astype(np.float64) * ts[:, None] * 6 >= a * (1 - 2.0 ** -4)).all()
    n = np.linalg.norm
    e1 = n(pp["A0"].astype(np.float64) - Xf) / n(Xf)
    e2 = n(pp["A0"].astype(np.float64) + pp["A1"].astype(np.float64) - Xf) / n(Xf)
    assert e2 < e1 / 4


@pytest.mark.parametrize("fmt", [so.NVFP4, so.MXFP4])
def test_sparse_sparse_paths_and_table5_ordering(fmt):
    """Sparse+Sparse: first path == SharQ's backbone bit for bit; the second mask is an exact top-2-of-4 on |R|
    (brute force), its survivors are exactly N of M; and the reconstruction errors order as Table 5 does:
    Sparse >> Sparse+Sparse > SharQ, Dense+Dense ~ SharQ."""
    x = si.activations(16, 2048, config=1); g = si.gamma(2048)
    ps = so.prepare_paths(x, so.PATH_SPARSE_SPARSE, fmt=fmt, gamma_u16=g)
    p = so.prepare(x, fmt=fmt, gamma_u16=g)
    for k0, k1 in (("a0_codes", "sp_codes"), ("a0_sf", "sp_sf"), ("a0_meta", "sp_meta")):
        assert np.array_equal(ps[k0], p[k1])
    assert np.array_equal(ps["R"], p["R"])
    keep1, nib1 = so.mask_pair48_f32(ps["R"])
    assert (keep1.reshape(16, -1, 8).sum(-1) == 4).all()
    score = np.abs(ps["R"]).reshape(16, -1, 4, 2).max(-1)
    for t in range(2):
        for c in range(score.shape[1]):
            best = _best_mask_bruteforce(score[t, c].tolist())
            assert nib1[t, c] == best[0] | (best[1] << 2)
    assert (ps["A1"][~keep1] == 0).all()
    # stored operands decode to A0 / A1 (linear_paths sees what the kernels see)
    w = si.weight(64, 2048); wq = so.quantize_weight(w, fmt)
    Wd = so.dequant_weight(wq)
    Y = so.linear_paths(ps, wq)
    # (A0 / A1 carry s_eff = RN(sf * ts) in fp32, the stored operands the exact product: 2^-24 relative per term)
    assert np.allclose(Y, (ps["A0"].astype(np.float64) + ps["A1"].astype(np.float64)) @ Wd.T, rtol=1e-6,
                       atol=1e-6 * np.abs(Y).max())
    Xf = so.bf16_to_f32(p["X"]).astype(np.float64)
    n = np.linalg.norm
    e_sparse = n(p["Xsp_tilde"].astype(np.float64) - Xf) / n(Xf)
    e_ss = n(ps["A0"].astype(np.float64) + ps["A1"].astype(np.float64) - Xf) / n(Xf)
    e_sharq = n(so.dequant_backbone(p) + so.dequant_residual(p) - Xf) / n(Xf)
    pd = so.prepare_paths(x, so.PATH_DENSE_DENSE, fmt=fmt, gamma_u16=g)
    e_dd = n(pd["A0"].astype(np.float64) + pd["A1"].astype(np.float64) - Xf) / n(Xf)
    assert e_sparse > 3 * e_ss > 3 * e_sharq and e_dd < 1.5 * e_sharq
    Yd = so.linear_paths(pd, wq)
    assert np.allclose(Yd, (pd["A0"].astype(np.float64) + pd["A1"].astype(np.float64)) @ Wd.T, rtol=1e-6,
                       atol=1e-6 * np.abs(Yd).max())


# ------------------------------------------------------------------ SwiGLU contract (R18)
def test_exp_contract_against_math_exp_and_special_values():
    """exp_neg_contract(g) ~= exp(-g): constants are RN of their definitions, relative error <= 3e-6 against
    math.exp over the whole useful range, exact at g = 0 and at g = -k ln 2 up to the rounding of t."""
    assert so.NEG_LOG2E == F32(-math.log2(math.e))
    for k in range(6):
        assert so.EXP2_POLY[k] == F32(math.log(2.0) ** k / math.factorial(k)), k
    assert so.exp_neg_contract(np.zeros(3, F32)).tolist() == [1.0, 1.0, 1.0]
    g = np.concatenate([np.linspace(-80, 80, 20001), np.random.default_rng(0).standard_normal(20000) * 8]).astype(F32)
    e = so.exp_neg_contract(g).astype(np.float64)
    ref = np.array([math.exp(-float(v)) for v in g])
    # degree-5 remainder 2.4e-6 + roundings; + the rounding of the constant log2e and of t = g * log2e (each up to
    # |g| 2^-24 relative in e)
    bound = 3.5e-6 + np.abs(g.astype(np.float64)) * 1.3e-7
    assert (np.abs(e - ref) <= bound * ref).all(), float((np.abs(e - ref) / ref / bound).max())
    # monotone non-increasing in g on a fine grid (a sign or index slip in the reduction would break it)
    gs = np.sort(g)
    es = so.exp_neg_contract(gs)
    assert (np.diff(es.astype(np.float64)) <= 2e-6 * es[:-1]).all()
    # clamp: no inf / nan at the ends, limits of the sigmoid
    big = so.exp_neg_contract(np.array([-1e4, 1e4], F32))
    assert np.isfinite(big).all() and big[0] >= 2.0 ** 125 and big[1] <= 2.0 ** -125


def test_swiglu_against_fp64_definition():
    """h = bf16(silu(g) * u): always one of the two bf16 neighbours of the exact value, equal to its RNE whenever the
    exact value is not within 1e-5 (relative) of a rounding boundary; exact special cases by hand."""
    rng = np.random.default_rng(1)
    g = so.f32_to_bf16((rng.standard_normal(200000) * 4).astype(F32))
    u = so.f32_to_bf16((rng.standard_normal(200000) * 2).astype(F32))
    h = so.bf16_to_f32(so.swiglu(g, u)).astype(np.float64)
    gf, uf = so.bf16_to_f32(g).astype(np.float64), so.bf16_to_f32(u).astype(np.float64)
    exact = gf / (1.0 + np.exp(-gf)) * uf
    rne = so.bf16_to_f32(so.f32_to_bf16(exact.astype(F32))).astype(np.float64)
    ulp = 2.0 ** (np.floor(np.log2(np.maximum(np.abs(exact), 1e-300))) - 7)
    assert (np.abs(h - exact) <= ulp * (0.5 + 1e-3) + 1e-38).all()               # a neighbour of the exact value
    away = np.abs(np.abs(exact - rne) - ulp / 2) > 2e-5 * np.abs(exact)           # not near a tie of the bf16 grid
    assert (h[away] == rne[away]).all()
    assert away.mean() > 0.99
    # by hand: g = 0 -> silu = 0; g = 40 -> sigmoid = 1 exactly in fp32 -> h = bf16(40 u); g = -40 -> ~ -40 e^-40 u
    hh = so.bf16_to_f32(so.swiglu(so.f32_to_bf16(np.array([0.0, 40.0, -40.0, 1.0], F32)),
                                  so.f32_to_bf16(np.array([3.0, 1.5, 2.0, 1.0], F32))))
    assert hh[0] == 0.0 and hh[1] == 60.0
    assert abs(hh[2] / (-40 * math.exp(-40) * 2.0) - 1) < 2.0 ** -8
    assert hh[3] == so.bf16_to_f32(so.f32_to_bf16(np.array([1 / (1 + math.exp(-1))], F32)))[0]
