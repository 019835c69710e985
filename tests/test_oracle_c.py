"""Cross-pin of the two oracles (not gpu): oracle/sharq_oracle_c.c and oracle/sharq_oracle.py are two independent
restatements of the same specification (the paper + DESIGN.md R1-R8).  Every stored output must agree byte for byte,
the fp64 linear to rounding-order noise.  A mistake in either one (a dropped term, a wrong tie rule, a transposed index)
has to be made identically in both languages to survive this file.  P:n = /root/reference/PAPER.md line n."""
import numpy as np
import pytest

import sharq_inputs as si
from oracle import c_oracle as co
from oracle import sharq_oracle as so

KEYS = ("sp_codes", "sp_sf", "sp_meta", "dn_codes", "dn_sf", "ts", "X")


def _same(pc, pn):
    for k in KEYS:
        a, b = pc[k], pn[k]
        assert a.shape == b.shape and a.dtype == b.dtype, k
        assert np.array_equal(a.view(np.uint8), b.view(np.uint8)), k


@pytest.mark.parametrize("fmt", [so.NVFP4, so.MXFP4])
@pytest.mark.parametrize("norm", [so.NORM_NONE, so.NORM_RMS, so.NORM_LAYER])
@pytest.mark.parametrize("K", [256, 1024, 3584])
def test_prepare_agrees_byte_for_byte(fmt, norm, K):
    T = 13
    x = si.activations(T, K, config=2, extra=K + norm)
    x[3] = 0                                                  # an all-zero row: ts = 1, every scale 0
    x[5, 8:16] = x[5, 0:8]                                     # equal scores across chunks
    x[6, :64] = si.to_bf16_bits(np.full(64, 0.75, np.float32)) # every pair ties: lower index wins
    g, b = si.gamma(K, 2), si.beta(K, 2)
    pc = co.prepare(x, fmt, norm, g, b if norm == so.NORM_LAYER else None, eps=1e-5)
    pn = so.prepare(x, fmt=fmt, norm=norm, gamma_u16=g, beta_u16=b if norm == so.NORM_LAYER else None, eps=1e-5)
    _same(pc, pn)


def test_canonical_sum_order_agrees():
    # R1: wide dynamic range makes every change of the addition order visible in the last bits
    rng = np.random.default_rng(11)
    differs_from_naive = 0
    for K in (256, 1000, 1024, 3584, 4096, 5000):
        for trial in range(20):
            t = (rng.standard_normal(K) * np.exp2(rng.integers(-12, 13, K))).astype(np.float32)
            for sq in (False, True):
                a, b = co.canonical_sum(t, sq), so.canonical_sum(t[None, :], squares=sq)[0]
                assert a.tobytes() == np.float32(b).tobytes(), (K, trial, sq)
            differs_from_naive += float(co.canonical_sum(t, False)) != float(np.cumsum(t, dtype=np.float32)[-1])
    assert differs_from_naive > 20                             # the inputs do discriminate between orders


def test_prepare_static_tensor_scale_and_threads():
    T, K = 9, 512
    x = si.activations(T, K, config=3)
    pn = so.prepare(x, norm=so.NORM_NONE, x_tensor_scale=0.004)
    for nt in (1, 3):
        pc = co.prepare(x, co.NVFP4, co.NORM_NONE, x_tensor_scale=0.004, nthreads=nt)
        assert pc["threads"] == nt
        _same(pc, pn)


def test_prepare_extreme_magnitudes():
    # scale codes at both ends: subnormal e4m3 scales, saturation, e8m0 clamps
    rng = np.random.default_rng(5)
    T, K = 6, 256
    base = rng.standard_normal((T, K)).astype(np.float32)
    mags = np.array([1e-30, 1e-12, 1e-3, 1.0, 1e12, 1e30], np.float32)[:, None]
    x = si.to_bf16_bits(base * mags)
    for fmt in (so.NVFP4, so.MXFP4):
        _same(co.prepare(x, fmt, co.NORM_NONE), so.prepare(x, fmt=fmt, norm=so.NORM_NONE))
    # one huge outlier per row next to tiny values: block scales underflow to zero for NVFP4
    x2 = si.to_bf16_bits(base * np.float32(1e-6))
    x2[:, 7] = si.to_bf16_bits(np.full(T, 3e4, np.float32))
    _same(co.prepare(x2, so.NVFP4, co.NORM_NONE), so.prepare(x2, fmt=so.NVFP4, norm=so.NORM_NONE))


@pytest.mark.parametrize("fmt", [so.NVFP4, so.MXFP4])
def test_weights_and_linear_agree(fmt):
    T, K, D = 7, 768, 40
    x, g, w = si.activations(T, K, config=4), si.gamma(K, 4), si.weight(D, K, 4)
    wc, wn = co.quantize_weight(w, fmt), so.quantize_weight(w, fmt=fmt)
    for k in ("codes", "sf_sp", "sf_dn"):
        assert np.array_equal(wc[k], wn[k]), k
    assert np.float32(wc["ts_w"]).tobytes() == np.float32(wn["ts_w"]).tobytes()
    pc, pn = co.prepare(x, fmt, co.NORM_RMS, g), so.prepare(x, fmt=fmt, norm=so.NORM_RMS, gamma_u16=g)
    Yc, Yn = co.linear(pc, wc), so.linear(pn, wn)
    scale = np.sqrt((Yn ** 2).mean())
    assert np.abs(Yc - Yn).max() <= 1e-12 * scale
    rows, cols = np.array([5, 0, 2]), np.array([39, 1, 17, 8])
    Ys = co.linear(pc, wc, rows=rows, cols=cols, nthreads=2)
    assert np.array_equal(Ys, Yc[np.ix_(rows, cols)])         # same order of additions: bit-identical
    assert abs(Yc[2, 17] - so.linear_loops(pn, wn, 2, 17)) <= 1e-12 * scale


def test_codec_tables_exhaustive():
    # every e4m3 / e8m0 / e2m1 decision on a dense sweep of inputs, through one block each: a block whose maximum is
    # the probe value exposes the scale code; the element codes expose e2m1 rounding at that scale
    vals = np.concatenate([np.linspace(0, 7, 449, dtype=np.float32), np.ldexp(np.float32(1), np.arange(-20, 12))])
    x = np.zeros((len(vals), 256), np.float32)
    x[:, 0] = vals
    x[:, 1] = vals * np.float32(0.4375)
    x[:, 2] = -vals * np.float32(0.3125)
    x[:, 32] = 1.0                                             # pins the row maximum's order of magnitude
    xb = si.to_bf16_bits(x)
    for fmt in (so.NVFP4, so.MXFP4):
        _same(co.prepare(xb, fmt, co.NORM_NONE, x_tensor_scale=None if fmt else 1.0 / 512),
              so.prepare(xb, fmt=fmt, norm=so.NORM_NONE, x_tensor_scale=None if fmt else 1.0 / 512))


def test_front_end_operators_agree():
    # N1 (R18): the residual-stream add and SiLU(gate) * up, bit for bit; the exp contract on a sweep incl. both clamps
    rng = np.random.default_rng(23)
    x = si.to_bf16_bits((rng.standard_normal(5000) * np.exp2(rng.integers(-20, 8, 5000))).astype(np.float32))
    r = si.to_bf16_bits((rng.standard_normal(5000) * np.exp2(rng.integers(-20, 8, 5000))).astype(np.float32))
    assert np.array_equal(co.residual_add(x, r), so.residual_add(x, r))
    g = si.to_bf16_bits(np.concatenate([np.linspace(-100, 100, 4001), rng.standard_normal(4000) * 4]).astype(np.float32))
    u = si.to_bf16_bits(rng.standard_normal(g.size).astype(np.float32))
    assert np.array_equal(co.swiglu(g, u), so.swiglu(g, u))
    assert np.array_equal(co.swiglu(g, u, nthreads=1), so.swiglu(g, u))
    for v in (-200.0, -88.0, -1.0, -1e-8, 0.0, 0.5, 17.3, 87.3, 88.0, 200.0):
        assert co.exp_neg(v).tobytes() == np.float32(so.exp_neg_contract(np.float32(v))).tobytes(), v


@pytest.mark.parametrize("norm", [so.NORM_NONE, so.NORM_RMS, so.NORM_LAYER])
@pytest.mark.parametrize("K", [256, 768, 3584])
def test_hif4_prepare_agrees_byte_for_byte(norm, K):
    # Algorithm 1, 2:4 mask, residual: every stored byte, incl. zero rows, ties, 1e-30 .. 1e30 magnitudes
    T = 12
    x = si.activations(T, K, config=2, outlier_mult=200.0, extra=K + norm)
    x[2] = 0
    x[3, :64] = si.to_bf16_bits(np.full(64, -0.75, np.float32))
    xf = si.bf16_bits_to_f32(x).copy()
    xf[4] *= 1e-30; xf[5] *= 1e30; xf[6] *= 2.0 ** -50; xf[7] *= 2.0 ** 14
    x = si.to_bf16_bits(xf) if norm == so.NORM_NONE else x
    g, b = si.gamma(K, 2), si.beta(K, 2)
    pc = co.prepare_hif4(x, norm, g, b if norm == so.NORM_LAYER else None, eps=1e-5)
    pn = so.prepare(x, fmt=so.HIF4, mask=so.MASK_24, norm=norm, gamma_u16=g, beta_u16=b if norm == so.NORM_LAYER else None,
                    eps=1e-5)
    for k in ("sp_meta", "sp_codes", "sp_sf", "dn_codes", "dn_sf"):
        assert pc[k].dtype == pn[k].dtype and np.array_equal(pc[k], pn[k]), k


def test_hif4_weights_and_linear_agree():
    T, K, D = 6, 512, 24
    x, g, w = si.activations(T, K, config=4), si.gamma(K, 4), si.weight(D, K, 4)
    wc, wn = co.quantize_weight_hif4(w), so.quantize_weight(w, fmt=so.HIF4)
    assert np.array_equal(wc["codes"], wn["codes"]) and np.array_equal(wc["sf_sp"], wn["sf_sp"])
    pc = co.prepare_hif4(x, so.NORM_RMS, g)
    pn = so.prepare(x, fmt=so.HIF4, mask=so.MASK_24, norm=so.NORM_RMS, gamma_u16=g)
    Yc, Yn = co.linear_hif4(pc, wc), so.linear(pn, wn)
    assert np.abs(Yc - Yn).max() <= 1e-12 * np.sqrt((Yn ** 2).mean())
    rows, cols = np.array([4, 1]), np.array([23, 0, 7])
    assert np.array_equal(co.linear_hif4(pc, wc, rows=rows, cols=cols, nthreads=2), Yc[np.ix_(rows, cols)])


def test_hif4_scale_codec_sweep():
    # every E6M2 rounding decision: units whose maximum sweeps 7 * (a fine grid over three octaves and both clamps)
    vals = np.concatenate([np.linspace(1.0, 8.0, 1793), [2.0 ** -60, 2.0 ** -49, 2.0 ** -48, 1.2 * 2.0 ** 17, 1e37]]).astype(np.float32)
    x = np.zeros((len(vals), 256), np.float32)
    x[:, 0] = vals * 7
    x[:, 1] = -vals * 3.3
    x[:, 5] = vals * 0.9
    x[:, 70] = vals
    xb = si.to_bf16_bits(x)
    pc, pn = co.prepare_hif4(xb, so.NORM_NONE), so.prepare(xb, fmt=so.HIF4, mask=so.MASK_24, norm=so.NORM_NONE)
    for k in ("sp_meta", "sp_codes", "sp_sf", "dn_codes", "dn_sf"):
        assert np.array_equal(pc[k], pn[k]), k


def test_rejects_bad_arguments():
    x = np.zeros((2, 100), np.uint16)
    with pytest.raises(ValueError):
        co.prepare(x, co.NVFP4, co.NORM_NONE)                 # K % 256
    with pytest.raises(ValueError):
        co.prepare(np.zeros((2, 256), np.uint16), co.NVFP4, co.NORM_RMS)   # gamma missing
