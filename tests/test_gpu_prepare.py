"""GPU parity: sharq_prepare and sharq_quantize_weight through the C ABI vs the oracle, bit-exact
(masks/metadata, packed codes, scale bytes, row scales).  BASELINE.json: "must match bit-exactly"."""
import numpy as np
import pytest
import torch

import sharq_inputs as si
from oracle import sharq_oracle as so
from tests.gpu_util import act_to_canonical, to_dev, weight_to_canonical

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sq():
    import __graft_entry__ as g
    g.build()
    import paper_2606_26587_b200 as pkg
    return pkg


def _compare_act(got, p, what=""):
    for key in ("sp_meta", "sp_sf", "sp_codes", "dn_sf", "dn_codes"):
        eq = got[key] == p[key]
        assert eq.all(), f"{what} {key}: {np.count_nonzero(~eq)} of {eq.size} differ, first at {np.argwhere(~eq)[:3].tolist()}"
    assert np.array_equal(got["ts"].view(np.uint32), p["ts"].view(np.uint32)), f"{what} row_scale"


CASES = [
    # (fmt, norm, layout, T, K, outlier_mult)   K spans several 1024-blocks and ragged tails (768, 3584)
    (0, 1, 0, 16, 4096, 50.0), (0, 1, 1, 16, 4096, 50.0), (0, 0, 1, 37, 14336, 50.0), (0, 1, 0, 5, 768, 10.0),
    (0, 1, 1, 130, 3584, 200.0), (0, 2, 0, 9, 2048, 50.0), (0, 0, 0, 1, 256, 50.0), (0, 1, 0, 300, 1024, 50.0),
    (1, 1, 0, 16, 4096, 50.0), (1, 0, 1, 33, 3584, 200.0), (1, 2, 0, 7, 768, 10.0), (1, 1, 1, 129, 18944, 50.0),
    (2, 1, 0, 16, 4096, 50.0), (2, 0, 0, 33, 3584, 200.0), (2, 2, 0, 7, 768, 10.0), (2, 1, 0, 3, 18944, 50.0),
    # the widest row one CTA covers (32 warps) and the first K beyond it (warp-per-row kernel, row in smem)
    (0, 1, 1, 3, 32768, 50.0), (0, 1, 1, 3, 33792, 50.0), (0, 2, 0, 150, 33792, 50.0), (1, 0, 0, 2, 33792, 200.0),
    (0, 2, 1, 5, 32768, 50.0), (0, 2, 0, 4, 25600, 50.0), (0, 2, 0, 4, 26624, 50.0),   # NVFP4 + LayerNorm around the one-CTA shared-memory limit
    (2, 1, 0, 2, 33792, 50.0),
]


@pytest.mark.parametrize("fmt,norm,layout,T,K,mult", CASES)
def test_prepare_bit_exact(sq, fmt, norm, layout, T, K, mult):
    x = si.activations(T, K, config=1, outlier_mult=mult, extra=K + T)
    g, b = si.gamma(K, 1), si.beta(K, 1)
    cfg = sq.make_config(fmt, norm, 1e-6, layout)
    act = sq.prepare(cfg, to_dev(x), to_dev(g) if norm else None, to_dev(b) if norm == 2 else None)
    torch.cuda.synchronize()
    p = so.prepare(x, fmt=fmt, mask=cfg.mask, norm=norm, gamma_u16=g, beta_u16=b if norm == 2 else None)
    _compare_act(act_to_canonical(sq, cfg, act, T, K), p, f"fmt{fmt} norm{norm} T{T} K{K}")


def test_prepare_edge_cases(sq):
    """zero rows, -0 / tiny values, exact ties, huge dynamic range, static tensor scale, strided input."""
    T, K = 12, 1024
    x = si.activations(T, K, config=1)
    xf = si.bf16_bits_to_f32(x).copy()
    xf[0] = 0.0
    xf[1] = -0.0
    xf[2] = 1.0                                   # every pair ties
    xf[3, ::2] = -3.0; xf[3, 1::2] = 3.0
    xf[4] *= 1e-30
    xf[5] *= 1e30
    xf[6, :512] = 0.0
    xf[7] = np.where(np.arange(K) % 8 < 4, 5.0, -5.0)
    x = si.to_bf16_bits(xf)
    x[1] = 0x8000
    for fmt in (0, 1, 2):
        cfg = sq.make_config(fmt, sq.NORM_NONE, 1e-6, sq.LAYOUT_CANONICAL)
        act = sq.prepare(cfg, to_dev(x))
        p = so.prepare(x, fmt=fmt, mask=cfg.mask, norm=so.NORM_NONE)
        _compare_act(act_to_canonical(sq, cfg, act, T, K), p, f"edge fmt{fmt}")
    # static per-tensor scale through a device pointer
    cfg = sq.make_config(0, sq.NORM_RMS, 1e-6, sq.LAYOUT_CANONICAL)
    g = si.gamma(K, 1)
    ts = torch.tensor([0.0078125], dtype=torch.float32, device="cuda")
    act = sq.prepare(cfg, to_dev(x), to_dev(g), x_tensor_scale=ts)
    p = so.prepare(x, gamma_u16=g, x_tensor_scale=0.0078125)
    _compare_act(act_to_canonical(sq, cfg, act, T, K), p, "static ts")
    # leading dimension > K
    big = torch.zeros((T, K + 64), dtype=torch.bfloat16, device="cuda")
    big[:, :K] = to_dev(x)
    act = sq.prepare(cfg, big[:, :K], to_dev(g))
    p = so.prepare(x, gamma_u16=g)
    _compare_act(act_to_canonical(sq, cfg, act, T, K), p, "ldx")


@pytest.mark.parametrize("fmt,layout,D,K", [(0, 0, 256, 4096), (0, 1, 384, 3584), (1, 1, 128, 768), (1, 0, 200, 1024),
                                            (2, 0, 256, 4096), (2, 0, 64, 768)])
def test_quantize_weight_bit_exact(sq, fmt, layout, D, K):
    w = si.weight(D, K, config=1, extra=D)
    cfg = sq.make_config(fmt, sq.NORM_NONE, 1e-6, layout)
    wq = sq.quantize_weight(cfg, to_dev(w))
    torch.cuda.synchronize()
    ref = so.quantize_weight(w, fmt)
    got = weight_to_canonical(sq, cfg, wq, D, K)
    for key in ("codes", "sf_sp") + (("sf_dn",) if fmt != 2 else ()):
        assert np.array_equal(got[key], ref[key]), key
    if fmt == 2:      # the GEMM-side view of a HiF4 payload is its exact bf16 dequantisation (Eq. 15)
        w64 = so.dequant_weight(ref)
        assert np.array_equal(so.bf16_to_f32(got["w_bf16"]).astype(np.float64), w64)
    assert np.float32(got["ts_w"]) == ref["ts_w"]


def test_prepare_full_size_sampled_rows(sq):
    """BASELINE configs[2] size (T=4096, K=4096 and K=14336) in the bench launch configuration: the
    oracle recomputes a seeded sample of rows (rows are independent)."""
    for (T, K, norm) in ((4096, 4096, 1), (2048, 14336, 0)):
        x = si.activations(T, K, config=3, outlier_mult=200.0)
        g = si.gamma(K, 3)
        cfg = sq.make_config(0, norm, 1e-6, sq.LAYOUT_TILED)
        act = sq.prepare(cfg, to_dev(x), to_dev(g) if norm else None)
        torch.cuda.synchronize()
        got = act_to_canonical(sq, cfg, act, T, K)
        rows = np.random.default_rng(T + K).choice(T, 48, replace=False)
        rows[:3] = (0, T - 1, T // 2)
        p = so.prepare(x[rows], norm=norm, gamma_u16=g)
        _compare_act({k: v[rows] for k, v in got.items()}, p, f"full T{T} K{K}")


@pytest.mark.parametrize("T,K,norm,static_ts,layout", [
    (3000, 9216, 1, None, 1),        # 9 warps per row: lagged loop, RMSNorm, 3 rows per CTA
    (2500, 18944, 2, None, 0),       # 19 warps, LayerNorm, canonical layout, 5-6 rows per CTA
    (2500, 14336, 0, 0.0625, 1),     # lagged loop without the row-amax exchange (static tensor scale)
    (5000, 8192, 1, None, 1),        # 8 warps: the widest row of the blocking loop, several rows per CTA
    (500, 32768, 1, None, 1),        # 32 warps (the widest one-CTA row), lagged loop, two rows in most CTAs
])
def test_prepare_many_rows_per_cta_sampled(sq, T, K, norm, static_ts, layout):
    """More rows than CTAs, so every CTA runs several iterations of the software-pipelined row loop (next row
    fetched inside the tail; for K > 8192 the lagged loop whose row-amax exchange is waited for one iteration
    later).  Rows are independent: the oracle recomputes a seeded sample, first and last rows included."""
    x = si.activations(T, K, config=2, outlier_mult=50.0, extra=T + K)
    g, b = si.gamma(K, 2), si.beta(K, 2)
    cfg = sq.make_config(0, norm, 1e-6, layout)
    ts = None if static_ts is None else torch.tensor([static_ts], dtype=torch.float32, device="cuda")
    act = sq.prepare(cfg, to_dev(x), to_dev(g) if norm else None, to_dev(b) if norm == 2 else None, x_tensor_scale=ts)
    torch.cuda.synchronize()
    got = act_to_canonical(sq, cfg, act, T, K)
    rows = np.random.default_rng(T + K).choice(T, 40, replace=False)
    rows[:4] = (0, 1, T - 1, T - 2)
    p = so.prepare(x[rows], norm=norm, gamma_u16=g if norm else None, beta_u16=b if norm == 2 else None,
                   x_tensor_scale=static_ts)
    _compare_act({k: v[rows] for k, v in got.items()}, p, f"T{T} K{K} norm{norm}")
    # rows outside the sample: every pair-4:8 metadata nibble is one of the six valid codes (no stale tile bytes)
    nib = np.concatenate([got["sp_meta"] & 0xF, got["sp_meta"] >> 4], axis=1)
    assert np.isin(nib, [0x4, 0x8, 0xC, 0x9, 0xD, 0xE]).all()


@pytest.mark.parametrize("fmt,norm,T,K,inplace", [
    (0, 1, 16, 4096, True),          # configs[0] shape: residual add + RMSNorm, in-place stream update
    (0, 1, 2100, 4096, False),       # several rows per CTA, blocking loop
    (0, 2, 700, 14336, True),        # lagged loop, LayerNorm
    (1, 1, 33, 3584, False),         # MXFP4, ragged K
    (2, 0, 9, 768, True),            # HiF4, no norm
])
def test_prepare_add_bit_exact(sq, fmt, norm, T, K, inplace):
    """sharq_prepare_add: the new residual stream equals the oracle's bf16(x + r) bit for bit and
    every prepared output equals the oracle's preparation of that sum."""
    x = si.activations(T, K, config=4, outlier_mult=50.0, extra=T)
    r = si.activations(T, K, config=5, outlier_mult=10.0, extra=K)
    g, b = si.gamma(K, 4), si.beta(K, 4)
    cfg = sq.make_config(fmt, norm, 1e-6, sq.LAYOUT_CANONICAL if fmt == 2 else sq.LAYOUT_TILED)
    xd, rd = to_dev(x), to_dev(r)
    out = None if inplace else torch.empty_like(rd)
    act, h_dev = sq.prepare_add(cfg, xd, rd, to_dev(g) if norm else None, to_dev(b) if norm == 2 else None, sum_out=out)
    torch.cuda.synchronize()
    h = so.residual_add(x, r)
    assert np.array_equal(h_dev.view(torch.int16).cpu().numpy().view(np.uint16), h), "residual stream"
    if not inplace:
        assert np.array_equal(rd.view(torch.int16).cpu().numpy().view(np.uint16), r), "residual input was modified"
    rows = np.arange(T) if T * K <= 600_000 else np.unique(np.r_[0, 1, T - 1, np.random.default_rng(T).choice(T, 40, replace=False)])
    p = so.prepare(h[rows], fmt=fmt, mask=cfg.mask, norm=norm, gamma_u16=g if norm else None, beta_u16=b if norm == 2 else None)
    got = act_to_canonical(sq, cfg, act, T, K)
    _compare_act({k: v[rows] for k, v in got.items()}, p, f"add fmt{fmt} norm{norm} T{T} K{K}")


def test_prepare_rows_not_32_byte_aligned(sq):
    """The C ABI asks for 16-byte alignment only; the row kernel reads 32 bytes per load, so rows that start on an
    odd 16-byte boundary are served by the warp-per-row kernel.  Same bytes out."""
    T, K = 19, 2048
    x = si.activations(T, K, config=1, extra=7)
    g = si.gamma(K, 1)
    cfg = sq.make_config(0, sq.NORM_RMS, 1e-6, sq.LAYOUT_TILED)
    buf = torch.zeros((T * (K + 8) + 8,), dtype=torch.bfloat16, device="cuda")
    view = buf[8:].view(T, K + 8)[:, :K]                    # base + 16 bytes, ldx = K + 8
    view.copy_(to_dev(x))
    assert view.data_ptr() % 32 == 16
    act = sq.prepare(cfg, view, to_dev(g))
    torch.cuda.synchronize()
    p = so.prepare(x, gamma_u16=g)
    _compare_act(act_to_canonical(sq, cfg, act, T, K), p, "misaligned")
    with pytest.raises(sq.SharqError):
        sq.prepare_add(cfg, view, to_dev(x), to_dev(g))


@pytest.mark.parametrize("fmt,norm,T,K", [(0, 1, 16, 4096), (0, 0, 37, 3584), (1, 1, 9, 768), (1, 2, 5, 33792), (0, 2, 130, 1024)])
def test_prepare_mask24_on_e2m1_formats_bit_exact(sq, fmt, norm, T, K):
    """SHARQ_MASK_24 (element-wise 2:4, P:95 / P:124) with NVFP4 / MXFP4: accepted by sharq_prepare,
    canonical layout, metadata K/8 bytes per row; sharq_linear refuses it (no such FP4 MMA on B200)."""
    x = si.activations(T, K, config=1, outlier_mult=50.0, extra=3 * K + T)
    g, b = si.gamma(K, 1), si.beta(K, 1)
    cfg = sq.make_config(fmt, norm, 1e-6, sq.LAYOUT_CANONICAL, mask=sq.MASK_24)
    act = sq.prepare(cfg, to_dev(x), to_dev(g) if norm else None, to_dev(b) if norm == 2 else None)
    torch.cuda.synchronize()
    p = so.prepare(x, fmt=fmt, mask=so.MASK_24, norm=norm, gamma_u16=g, beta_u16=b if norm == 2 else None)
    assert p["sp_meta"].shape == (T, K // 8)
    _compare_act(act_to_canonical(sq, cfg, act, T, K), p, f"mask24 fmt{fmt} norm{norm} T{T} K{K}")
    w = sq.quantize_weight(sq.make_config(fmt, 0, 1e-6, sq.LAYOUT_CANONICAL, mask=sq.MASK_24), to_dev(si.weight(128, K, 1)))
    with pytest.raises(sq.SharqError) as e:
        sq.linear(cfg, act, w)
    assert e.value.status == sq.ESHAPE


def test_tiled_pad_rows_are_initialised(sq):
    """TILED scale / metadata buffers are padded to 128 rows; alloc_act -> sharq_act_init gives the pad rows valid
    operands (zero scales, metadata nibble 0x4) and sharq_prepare leaves them alone."""
    T, K = 5, 512
    cfg = sq.make_config(0, 0, 1e-6, sq.LAYOUT_TILED)
    act = sq.prepare(cfg, to_dev(si.activations(T, K, config=1)))
    torch.cuda.synchronize()
    sf = sq.untile_sf(act["sp_sf"], 128, K // 32).cpu().numpy()
    dn = sq.untile_sf(act["dn_sf"], 128, K // 16).cpu().numpy()
    meta = sq.untile_meta(act["sp_meta"], 128, K).cpu().numpy()
    assert (sf[T:] == 0).all() and (dn[T:] == 0).all() and (meta[T:] == 0x44).all()
    assert (meta[:T] != 0).all()


@pytest.mark.parametrize("fmt,T,K,halves", [(0, 16, 14336, True), (0, 700, 4096, False), (1, 33, 3584, True), (2, 9, 768, False),
                                            (0, 300, 18944, True)])
def test_prepare_swiglu_bit_exact(sq, fmt, T, K, halves):
    """sharq_prepare_swiglu: every prepared output equals the oracle's preparation of
    h = bf16(silu(gate) * up) computed by the restatable exp contract (R18); gate / up given as two tensors
    or as the two column halves of one [T, 2K] gate+up output."""
    g_bits = si.activations(T, K, config=4, outlier_mult=5.0, extra=T + 1)
    u_bits = si.activations(T, K, config=5, outlier_mult=50.0, extra=K + 2)
    g_bits[0, :8] = si.to_bf16_bits(np.array([0.0, -0.0, 40.0, -40.0, 100.0, -100.0, 1e-30, -88.0], np.float32))
    cfg = sq.make_config(fmt, sq.NORM_NONE, 1e-6, sq.LAYOUT_CANONICAL if fmt == 2 else sq.LAYOUT_TILED)
    if halves:
        both = torch.cat([to_dev(g_bits), to_dev(u_bits)], dim=1)
        gd, ud = both[:, :K], both[:, K:]
    else:
        gd, ud = to_dev(g_bits), to_dev(u_bits)
    act = sq.prepare_swiglu(cfg, gd, ud)
    torch.cuda.synchronize()
    h = so.swiglu(g_bits, u_bits)
    p = so.prepare(h, fmt=fmt, mask=cfg.mask, norm=so.NORM_NONE)
    _compare_act(act_to_canonical(sq, cfg, act, T, K), p, f"swiglu fmt{fmt} T{T} K{K}")
