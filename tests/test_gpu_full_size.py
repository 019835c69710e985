"""GPU parity at BASELINE.json's FULL sizes, every output byte: the compiled C oracle (oracle/sharq_oracle_c.c, held
byte-identical to the numpy oracle by tests/test_oracle_c.py) is fast enough to recompute whole tensors, so these cases
compare ALL rows of sharq_prepare / sharq_quantize_weight, and whole output rows of sharq_linear, in the launch
configuration bench.py times (TILED layout, headline shapes).  The sampled-row tests elsewhere stay: they run the numpy
oracle directly."""
import numpy as np
import pytest
import torch

import sharq_inputs as si
from oracle import c_oracle as co
from tests.gpu_util import act_to_canonical, to_dev, weight_to_canonical

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sq():
    import __graft_entry__ as g
    g.build()
    import paper_2606_26587_b200 as pkg
    return pkg


def _all_equal(got, ref, keys, what):
    for key in keys:
        eq = got[key] == ref[key]
        assert eq.all(), f"{what} {key}: {np.count_nonzero(~eq)} of {eq.size} differ, first at {np.argwhere(~eq)[:3].tolist()}"


@pytest.mark.parametrize("fmt,norm,T,K,mult", [
    (0, 1, 8192, 4096, 50.0),        # headline qkv / gate+up activation: RMSNorm, 8192 rows
    (0, 0, 8192, 14336, 200.0),      # headline down activation: 14 warps per row, lagged loop
    (1, 1, 4096, 3584, 50.0),        # configs[3] Qwen, MXFP4, ragged 1024-block
    (0, 2, 4096, 4096, 10.0),        # LayerNorm at prefill size
])
def test_prepare_full_tensor_every_byte(sq, fmt, norm, T, K, mult):
    x = si.activations(T, K, config=3, outlier_mult=mult, extra=T + K + fmt)
    g, b = si.gamma(K, 3), si.beta(K, 3)
    cfg = sq.make_config(fmt, norm, 1e-6, sq.LAYOUT_TILED)
    act = sq.prepare(cfg, to_dev(x), to_dev(g) if norm else None, to_dev(b) if norm == 2 else None)
    torch.cuda.synchronize()
    got = act_to_canonical(sq, cfg, act, T, K)
    ref = co.prepare(x, fmt, norm, g if norm else None, b if norm == 2 else None, eps=1e-6, want_X=False)
    _all_equal(got, ref, ("sp_meta", "sp_sf", "sp_codes", "dn_sf", "dn_codes"), f"fmt{fmt} norm{norm} T{T} K{K}")
    assert np.array_equal(got["ts"].view(np.uint32), ref["ts"].view(np.uint32))


@pytest.mark.parametrize("fmt,D,K", [(0, 6144, 4096), (0, 4096, 14336), (1, 4608, 3584)])
def test_quantize_weight_full_tensor_every_byte(sq, fmt, D, K):
    w = si.weight(D, K, config=3, extra=D + fmt)
    cfg = sq.make_config(fmt, sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
    wq = sq.quantize_weight(cfg, to_dev(w))
    torch.cuda.synchronize()
    got, ref = weight_to_canonical(sq, cfg, wq, D, K), co.quantize_weight(w, fmt)
    _all_equal(got, ref, ("codes", "sf_sp", "sf_dn"), f"weight fmt{fmt} D{D} K{K}")
    assert np.float32(got["ts_w"]).tobytes() == np.float32(ref["ts_w"]).tobytes()


@pytest.mark.parametrize("fmt,norm,T,K,D", [
    (0, 1, 8192, 4096, 6144),        # headline qkv: CTA-pair tiles
    (0, 0, 8192, 14336, 4096),       # headline down: long K
    (0, 0, 128, 4096, 4096),         # configs[1] decode o at T = 128
    (1, 1, 4096, 3584, 4608),        # configs[3] Qwen qkv, MXFP4
])
def test_linear_whole_rows_at_full_size(sq, fmt, norm, T, K, D):
    """Every output feature of 48 seeded rows (first / last rows of the first / last row blocks included): a tile-order,
    ragged-tile or epilogue-store mistake anywhere along D shows up, which a column sample could miss."""
    x, g, w = si.activations(T, K, config=3, extra=T + D), si.gamma(K, 3), si.weight(D, K, config=3, extra=D)
    cfg = sq.make_config(fmt, norm, 1e-6, sq.LAYOUT_TILED)
    wq = sq.quantize_weight(cfg, to_dev(w))
    act = sq.prepare(cfg, to_dev(x), to_dev(g) if norm else None)
    y = sq.linear(cfg, act, wq, out_dtype="fp32")
    torch.cuda.synchronize()
    rows = np.random.default_rng(T + D).choice(T, 48, replace=False)
    rows[:6] = (0, 1, 127, T - 128, T - 2, T - 1)
    rows = np.unique(rows)
    y64 = co.linear(co.prepare(x, fmt, norm, g if norm else None, want_X=False), co.quantize_weight(w, fmt), rows=rows)
    got = y[torch.from_numpy(rows).cuda()].cpu().numpy().astype(np.float64)
    err = np.abs(got - y64) / np.maximum(np.abs(y64), 1e-2 * np.sqrt((y64 ** 2).mean()))       # DESIGN.md R15
    assert err.max() <= 1e-3, (err.max(), np.unravel_index(err.argmax(), err.shape))


def test_prepare_add_full_tensor_every_byte(sq):
    """sharq_prepare_add at the size bench.py times (T = 8192, K = 4096, RMSNorm, in place): the whole new residual
    stream and every prepared byte."""
    T, K = 8192, 4096
    x = si.activations(T, K, config=4, outlier_mult=50.0, extra=T)
    r = si.activations(T, K, config=5, outlier_mult=10.0, extra=K)
    g = si.gamma(K, 4)
    cfg = sq.make_config(0, 1, 1e-6, sq.LAYOUT_TILED)
    act, h_dev = sq.prepare_add(cfg, to_dev(x), to_dev(r), to_dev(g))
    torch.cuda.synchronize()
    h = co.residual_add(x, r)
    assert np.array_equal(h_dev.view(torch.int16).cpu().numpy().view(np.uint16), h), "residual stream"
    ref = co.prepare(h, 0, 1, g, eps=1e-6, want_X=False)
    _all_equal(act_to_canonical(sq, cfg, act, T, K), ref, ("sp_meta", "sp_sf", "sp_codes", "dn_sf", "dn_codes"), "prepare_add")


def test_prepare_swiglu_full_tensor_every_byte(sq):
    """sharq_prepare_swiglu at the size bench.py times (T = 8192, K = 14336, gate / up as the halves of one [T, 2K]
    gate+up output): every prepared byte against the C oracle's restatement of the exp contract (R18)."""
    T, K = 8192, 14336
    g_bits = si.activations(T, K, config=4, outlier_mult=5.0, extra=T + 1)
    u_bits = si.activations(T, K, config=5, outlier_mult=50.0, extra=K + 2)
    cfg = sq.make_config(0, sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
    both = torch.cat([to_dev(g_bits), to_dev(u_bits)], dim=1)
    act = sq.prepare_swiglu(cfg, both[:, :K], both[:, K:])
    torch.cuda.synchronize()
    ref = co.prepare(co.swiglu(g_bits, u_bits), 0, 0, want_X=False)
    _all_equal(act_to_canonical(sq, cfg, act, T, K), ref, ("sp_meta", "sp_sf", "sp_codes", "dn_sf", "dn_codes"), "prepare_swiglu")
    assert np.array_equal(act_to_canonical(sq, cfg, act, T, K)["ts"].view(np.uint32), ref["ts"].view(np.uint32))


@pytest.mark.parametrize("norm,T,K", [(1, 4096, 3584), (0, 4096, 18944)])
def test_hif4_prepare_full_tensor_every_byte(sq, norm, T, K):
    """HiF4 sharq_prepare (packed bf16x2 Algorithm 1) at configs[3]'s sizes: every stored byte of every row against the
    C oracle's scalar restatement of Algorithm 1."""
    x, g = si.activations(T, K, config=4, outlier_mult=50.0, extra=T + K), si.gamma(K, 4)
    cfg = sq.make_config(sq.HIF4, norm, 1e-6, sq.LAYOUT_CANONICAL)
    act = sq.prepare(cfg, to_dev(x), to_dev(g) if norm else None)
    torch.cuda.synchronize()
    ref = co.prepare_hif4(x, norm, g if norm else None, eps=1e-6)
    _all_equal(act_to_canonical(sq, cfg, act, T, K), ref, ("sp_meta", "sp_sf", "sp_codes", "dn_sf", "dn_codes"), f"hif4 norm{norm} K{K}")


def test_hif4_weight_and_linear_whole_rows_at_full_size(sq):
    """configs[3] Qwen qkv in HiF4 (T = 4096, 3584 -> 4608): the whole weight payload byte for byte, its bf16 GEMM-side
    view equal to the decoded values, and every output feature of 40 seeded rows of the sparse + dense bf16 GEMM."""
    T, K, D = 4096, 3584, 4608
    x, g, w = si.activations(T, K, config=4, extra=T + D), si.gamma(K, 4), si.weight(D, K, config=4, extra=D)
    cfg = sq.make_config(sq.HIF4, 1, 1e-6, sq.LAYOUT_CANONICAL)
    wq = sq.quantize_weight(cfg, to_dev(w))
    act = sq.prepare(cfg, to_dev(x), to_dev(g))
    y = sq.linear(cfg, act, wq, out_dtype="fp32")
    torch.cuda.synchronize()
    wc = co.quantize_weight_hif4(w)
    got_w = weight_to_canonical(sq, cfg, wq, D, K)
    assert np.array_equal(got_w["codes"], wc["codes"]) and np.array_equal(got_w["sf_sp"], wc["sf_sp"])
    rows = np.random.default_rng(T + D).choice(T, 40, replace=False)
    rows[:6] = (0, 1, 127, T - 128, T - 2, T - 1)
    rows = np.unique(rows)
    y64 = co.linear_hif4(co.prepare_hif4(x, 1, g, eps=1e-6), wc, rows=rows)
    got = y[torch.from_numpy(rows).cuda()].cpu().numpy().astype(np.float64)
    err = np.abs(got - y64) / np.maximum(np.abs(y64), 1e-2 * np.sqrt((y64 ** 2).mean()))
    assert err.max() <= 1e-3, (err.max(), np.unravel_index(err.argmax(), err.shape))
