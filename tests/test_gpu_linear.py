"""GPU parity: sharq_linear / sharq_linear_grouped through the C ABI vs the oracle's fp64 product of the
same dequantized operands (Eq. 9).  Bar (BASELINE.json north_star, R15):
|Y - Y64| <= 1e-3 * max(|Y64|, 1e-2 * rms(Y64)) on the fp32 output; the bf16 output must be the RNE
rounding of the fp32 output bit for bit."""
import numpy as np
import pytest
import torch

import sharq_inputs as si
from oracle import sharq_oracle as so
from tests.gpu_util import to_dev

pytestmark = pytest.mark.gpu
TOL = 1e-3


@pytest.fixture(scope="module")
def sq():
    import __graft_entry__ as g
    g.build()
    import paper_2606_26587_b200 as pkg
    return pkg


def rel_err(y, y64):
    den = np.maximum(np.abs(y64), 1e-2 * np.sqrt((y64 ** 2).mean()))
    return np.abs(y.astype(np.float64) - y64) / den


def path_reference(p, q, path):
    """Table 5's ablation rows: 0 = sparse + dense, 1 = sparse only, 2 = dense only."""
    A_sp, A_dn = so.dequant_backbone(p, with_ts=False), so.dequant_residual(p, with_ts=False)
    W_sp, W_dn = so.dequant_weight(q, "sparse", with_ts=False), so.dequant_weight(q, "dense", with_ts=False)
    acc = (A_sp @ W_sp.T if path != 2 else 0.0) + (A_dn @ W_dn.T if path != 1 else 0.0)
    return acc * p["ts"].astype(np.float64)[:, None] * np.float64(q["ts_w"])


CASES = [
    # (fmt, norm, T, K, D, mult)   several k-blocks and n-tiles, ragged T (not a multiple of 128), T = 1
    (0, 1, 16, 4096, 4096, 50.0),      # BASELINE.json configs[0]
    (0, 1, 1, 4096, 6144, 50.0), (0, 0, 8, 14336, 4096, 50.0), (0, 1, 32, 4096, 28672, 50.0),   # configs[1] shapes
    (0, 1, 300, 1024, 384, 200.0), (0, 0, 129, 256, 128, 10.0), (0, 1, 257, 3584, 512, 50.0),
    (1, 1, 16, 4096, 4096, 50.0), (1, 0, 130, 3584, 4608, 200.0), (1, 1, 5, 768, 2048, 10.0),
    # HiF4: exact bf16 emulation path (128- and 256-wide tiles, ragged T)
    (2, 1, 16, 4096, 4096, 50.0), (2, 0, 130, 768, 384, 10.0), (2, 1, 300, 3584, 512, 200.0),
    (2, 0, 600, 768, 3328, 50.0),      # HiF4 CTA-pair bf16 tiles: 5 row blocks (ragged pair, ragged T) x 13 n-tiles
    (0, 1, 5, 33792, 256, 50.0),       # K beyond one prepare CTA; 132 k-blocks
]


@pytest.mark.parametrize("fmt,norm,T,K,D,mult", CASES)
def test_linear_vs_oracle(sq, fmt, norm, T, K, D, mult):
    x = si.activations(T, K, config=2, outlier_mult=mult, extra=T + K)
    g, w = si.gamma(K, 2), si.weight(D, K, 2, extra=D)
    cfg = sq.make_config(fmt, norm, 1e-6, sq.LAYOUT_TILED)
    wq = sq.quantize_weight(cfg, to_dev(w))
    act = sq.prepare(cfg, to_dev(x), to_dev(g) if norm else None)
    y32 = sq.linear(cfg, act, wq, out_dtype="fp32")
    y16 = sq.linear(cfg, act, wq, out_dtype="bf16")
    torch.cuda.synchronize()
    p = so.prepare(x, fmt=fmt, norm=norm, gamma_u16=g)
    q = so.quantize_weight(w, fmt=fmt)
    err = rel_err(y32.cpu().numpy(), so.linear(p, q))
    assert err.max() <= TOL, f"max rel err {err.max():.3e} at {np.unravel_index(err.argmax(), err.shape)}"
    assert torch.equal(y16, y32.to(torch.bfloat16)), "bf16 output is not RNE(fp32 output)"


@pytest.mark.parametrize("path", [1, 2])
def test_linear_single_path_and_bias(sq, path):
    T, K, D = 70, 1024, 256
    x, g, w = si.activations(T, K, config=3), si.gamma(K, 3), si.weight(D, K, 3)
    bias = si.beta(D, 3)
    cfg = sq.make_config(sq.NVFP4, sq.NORM_RMS, 1e-6, sq.LAYOUT_TILED)
    wq, act = sq.quantize_weight(cfg, to_dev(w)), sq.prepare(cfg, to_dev(x), to_dev(g))
    y = sq.linear(cfg, act, wq, out_dtype="fp32", path=path)
    yb = sq.linear(cfg, act, wq, bias=to_dev(bias), out_dtype="fp32", path=0)
    torch.cuda.synchronize()
    p, q = so.prepare(x, gamma_u16=g), so.quantize_weight(w)
    assert rel_err(y.cpu().numpy(), path_reference(p, q, path)).max() <= TOL
    assert rel_err(yb.cpu().numpy(), so.linear(p, q, bias_u16=bias)).max() <= TOL


def test_linear_strided_output_and_empty(sq):
    T, K, D = 9, 512, 256
    x, w = si.activations(T, K, config=3, extra=1), si.weight(D, K, 3, extra=1)
    cfg = sq.make_config(sq.NVFP4, sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
    wq, act = sq.quantize_weight(cfg, to_dev(w)), sq.prepare(cfg, to_dev(x))
    big = torch.full((T, D + 64), 7.0, dtype=torch.float32, device="cuda")
    sq.linear(cfg, act, wq, Y=big[:, :D])
    torch.cuda.synchronize()
    assert (big[:, D:] == 7.0).all(), "wrote outside the [T, D] window of a strided Y"
    p, q = so.prepare(x, norm=0), so.quantize_weight(w)
    assert rel_err(big[:, :D].cpu().numpy(), so.linear(p, q)).max() <= TOL
    # T = 0: SHARQ_OK, nothing launched, nothing touched
    empty = sq.alloc_act(cfg, 0, K, "cuda")
    y0 = sq.linear(cfg, empty, wq, Y=torch.empty((0, D), dtype=torch.float32, device="cuda"))
    assert y0.shape == (0, D)


def test_linear_rejects_bad_arguments(sq):
    cfg = sq.make_config(sq.NVFP4, sq.NORM_NONE, 1e-6, sq.LAYOUT_CANONICAL)
    x, w = si.activations(4, 256, config=3), si.weight(128, 256, 3)
    wq, act = sq.quantize_weight(cfg, to_dev(w)), sq.prepare(cfg, to_dev(x))
    with pytest.raises(sq.SharqError) as e:           # canonical layout is not what the GEMM consumes
        sq.linear(cfg, act, wq)
    assert e.value.status == sq.EINVAL


def test_linear_grouped_moe(sq):
    """Config 5 shape family, scaled down: experts with 0, 1, ragged and > 128 rows."""
    E, K, D = 6, 512, 256
    counts = [0, 1, 130, 37, 0, 128]
    offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    cfg = sq.make_config(sq.NVFP4, sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
    pad = [-(-c // 128) * 128 for c in counts]
    pad_off = np.concatenate([[0], np.cumsum(pad)])
    act = sq.alloc_act(cfg, int(pad_off[-1]), K, "cuda")
    ws, xs = [], []
    for e in range(E):
        ws.append(si.weight(D, K, 5, extra=e))
        xs.append(si.activations(counts[e], K, config=5, extra=e))
        if counts[e]:
            sq.prepare(cfg, to_dev(xs[e]), out=sq.act_slot(cfg, act, int(pad_off[e]), counts[e]))
    wqs = [sq.quantize_weight(cfg, to_dev(w)) for w in ws]
    wq = dict(codes=torch.cat([q["codes"] for q in wqs]), sf_sp=torch.cat([q["sf_sp"] for q in wqs]),
              sf_dn=torch.cat([q["sf_dn"] for q in wqs]), ts_w=torch.cat([q["ts_w"] for q in wqs]), D=D, K=K)
    Y = sq.linear_grouped(cfg, offsets, act, wq, D, out_dtype="fp32")
    torch.cuda.synchronize()
    Y = Y.cpu().numpy()
    for e in range(E):
        if counts[e] == 0:
            continue
        p, q = so.prepare(xs[e], norm=0), so.quantize_weight(ws[e])
        got = Y[pad_off[e]: pad_off[e] + counts[e]]
        assert rel_err(got, so.linear(p, q)).max() <= TOL, f"expert {e}"


def test_prefill_full_size_sampled(sq):
    """BASELINE.json configs[2] size, in the launch configuration bench.py times (CTA-pair 256x256 kernel,
    persistent over all SMs): T = 4096, K = 4096, D = 6144.  The oracle computes a seeded sample of rows
    (each row of prepare and linear is independent) and output features one by one."""
    T, K, D = 4096, 4096, 6144
    x, g, w = si.activations(T, K, config=3, outlier_mult=200.0), si.gamma(K, 3), si.weight(D, K, 3, extra=7)
    cfg = sq.make_config(sq.NVFP4, sq.NORM_RMS, 1e-6, sq.LAYOUT_TILED)
    wq = sq.quantize_weight(cfg, to_dev(w))
    act = sq.prepare(cfg, to_dev(x), to_dev(g))
    y32 = sq.linear(cfg, act, wq, out_dtype="fp32")
    y16 = sq.linear(cfg, act, wq, out_dtype="bf16")
    torch.cuda.synchronize()
    rng = np.random.Generator(np.random.Philox(si.seed_for(3, 99)))
    rows = np.sort(rng.choice(T, size=40, replace=False))
    rows[:4] = [0, 127, 128, T - 1]                       # tile corners
    rows = np.unique(rows)
    cols = np.unique(np.concatenate([rng.choice(D, size=250, replace=False), [0, 127, 128, 255, 256, D - 1]]))
    p = so.prepare(x[rows], gamma_u16=g)
    q = so.quantize_weight(w)
    # prepare outputs of the sampled rows, bit for bit (codes are row-major in both layouts)
    assert np.array_equal(act["sp_codes"].cpu().numpy().reshape(T, K // 4)[rows], p["sp_codes"])
    assert np.array_equal(act["dn_codes"].cpu().numpy().reshape(T, K // 2)[rows], p["dn_codes"])
    y64 = so.linear(p, q, cols=cols)
    got = y32.cpu().numpy()[np.ix_(rows, cols)]
    den = np.maximum(np.abs(y64), 1e-2 * np.sqrt((y64 ** 2).mean()))
    err = np.abs(got - y64) / den
    assert err.max() <= TOL, err.max()
    assert torch.equal(y16, y32.to(torch.bfloat16))


def test_moe_config5_size_sampled(sq):
    """BASELINE.json configs[4]: Qwen3-30B-A3B-shaped experts (gate+up 2048 -> 1536), 128 experts, seeded
    top-8 routing of 4096 tokens (0 .. ~600 rows per expert); three experts checked against the oracle."""
    E, K, D = 128, 2048, 1536
    ids, offsets, order = si.moe_routing()
    counts = np.diff(offsets)
    assert counts.sum() == 4096 * 8 and counts.min() >= 0
    cfg = sq.make_config(sq.NVFP4, sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
    pad_off = np.concatenate([[0], np.cumsum(-(-counts // 128) * 128)])
    act = sq.alloc_act(cfg, int(pad_off[-1]), K, "cuda")
    tokens = si.activations(4096, K, config=5)
    routed_token = (order // 8).astype(np.int64)            # token of every routed row, grouped by expert
    check = [int(np.argmax(counts)), int(np.argmin(counts)), 77]
    ws = {}
    wq_parts = []
    for e in range(E):
        w = si.weight(D, K, 5, extra=e) if e in check else si.weight(D, K, 5, extra=e % 3 + 1000)
        if e in check:
            ws[e] = w
        wq_parts.append(sq.quantize_weight(cfg, to_dev(w)))
        if counts[e]:
            xe = tokens[routed_token[offsets[e]: offsets[e + 1]]]
            sq.prepare(cfg, to_dev(xe), out=sq.act_slot(cfg, act, int(pad_off[e]), int(counts[e])))
    wq = dict(codes=torch.cat([q["codes"] for q in wq_parts]), sf_sp=torch.cat([q["sf_sp"] for q in wq_parts]),
              sf_dn=torch.cat([q["sf_dn"] for q in wq_parts]), ts_w=torch.cat([q["ts_w"] for q in wq_parts]), D=D, K=K)
    Y = sq.linear_grouped(cfg, offsets, act, wq, D, out_dtype="fp32")
    torch.cuda.synchronize()
    Y = Y.cpu().numpy()
    for e in check:
        if counts[e] == 0:
            continue
        xe = tokens[routed_token[offsets[e]: offsets[e + 1]]]
        y64 = so.linear(so.prepare(xe, norm=0), so.quantize_weight(ws[e]))
        got = Y[pad_off[e]: pad_off[e] + counts[e]]
        den = np.maximum(np.abs(y64), 1e-2 * np.sqrt((y64 ** 2).mean()))
        assert (np.abs(got - y64) / den).max() <= TOL, f"expert {e}"


def _sampled_check(sq, fmt, norm, T, K, D, config, mult, n_rows, n_cols, seed_extra):
    """Full-size launch, oracle on a seeded sample: prepare and linear are independent per activation row
     and per weight row (Eq. 9), except for the NVFP4 weight tensor scale max|W| / 2688,
    so the sampled weight rows always include the row that holds max|W|."""
    x, g, w = si.activations(T, K, config=config, outlier_mult=mult, extra=seed_extra), si.gamma(K, config), \
        si.weight(D, K, config, extra=seed_extra + 1)
    cfg = sq.make_config(fmt, norm, 1e-6, sq.LAYOUT_TILED)
    wq = sq.quantize_weight(cfg, to_dev(w))
    act = sq.prepare(cfg, to_dev(x), to_dev(g) if norm else None)
    y32 = sq.linear(cfg, act, wq, out_dtype="fp32")
    y16 = sq.linear(cfg, act, wq, out_dtype="bf16")
    torch.cuda.synchronize()
    rng = np.random.Generator(np.random.Philox(si.seed_for(config, 1000 + seed_extra)))
    last_blk = (T - 1) // 128 * 128                                # first row of the (possibly ragged) last 128-row block
    rows = np.unique(np.concatenate([rng.choice(T, size=min(n_rows, T), replace=False),
                                     [0, min(127, T - 1), min(128, T - 1), min(255, T - 1), min(256, T - 1),
                                      last_blk, max(last_blk - 1, 0), T - 1]]))
    w_mag = w & np.uint16(0x7FFF)                                  # bf16 magnitudes order like integers
    top_row = int(np.unravel_index(int(w_mag.argmax()), w_mag.shape)[0])
    # tile corners of the 128- / 192- / 256-wide variants and the tail of a ragged last N tile
    cols = np.unique(np.concatenate([rng.choice(D, size=n_cols, replace=False),
                                     [0, 127, 128, 191, 192, 255, 256, D - 64, D - 33, D - 2, D - 1, top_row]]))
    p = so.prepare(x[rows], fmt=fmt, norm=norm, gamma_u16=g)
    q = so.quantize_weight(w[cols], fmt=fmt)
    y64 = so.linear(p, q)
    got = y32.cpu().numpy()[np.ix_(rows, cols)]
    err = rel_err(got, y64)
    assert err.max() <= TOL, f"max rel err {err.max():.3e}"
    assert torch.equal(y16, y32.to(torch.bfloat16))


@pytest.mark.parametrize("T,K,D", [(256, 4096, 28672), (128, 4096, 28672), (100, 4096, 28672), (128, 14336, 4096), (256, 14336, 4096),
                                   (128, 4096, 6144)])
def test_decode_full_size_sampled(sq, T, K, D):
    """BASELINE.json configs[1] at its two largest token counts, in the launch configurations bench.py
    times there: CTA-pair tiles (T = 256), 128 x 256 tiles with full and ragged 128-row activation boxes,
    128-row split-K clusters and the persistent 128-wide kernel."""
    _sampled_check(sq, 0, 1 if K == 4096 else 0, T, K, D, config=2, mult=50.0, n_rows=24, n_cols=200,
                   seed_extra=T + D)


@pytest.mark.parametrize("fmt", [0, 1, 2])
def test_qwen_config4_full_size_sampled(sq, fmt):
    """BASELINE.json configs[3]: Qwen2.5-7B down projection 18944 -> 3584 at T = 4096 in all three formats
    (the longest K of the five configs: 74 k-blocks, ragged against every pipeline depth)."""
    _sampled_check(sq, fmt, 0, 4096, 18944, 3584, config=4, mult=50.0, n_rows=16, n_cols=120, seed_extra=fmt)


PREFILL_VARIANTS = [
    # (fmt, norm, T, K, D, mult)  every (shape, T, format) family bench.py times at prefill sizes, by launch variant
    (0, 0, 4096, 4096, 4096, 50.0),     # Llama o: CTA-pair tiles; 192-wide -> 22 n-tiles, ragged last (TMA zero fill)
    (0, 1, 4096, 4096, 28672, 50.0),    # Llama gate+up: 150 n-tiles of 192, ragged last
    (0, 0, 4096, 3584, 3584, 50.0),     # Qwen o: D % 256 != 0 -> 192-wide, 19 tiles, ragged last
    (0, 1, 4000, 4096, 6144, 50.0),     # pair kernel, ragged T: 32 row blocks, last one 32 rows
    (0, 1, 2049, 4096, 6144, 200.0),    # pair kernel, ODD number of 128-row blocks (17), last block one row
    (0, 0, 2177, 14336, 4096, 50.0),    # long K (256-wide by the cost model), ragged T
    (0, 0, 2048, 14336, 4096, 10.0),    # configs[2] T = 2048, outliers x10
    (0, 0, 8192, 14336, 4096, 200.0),   # configs[2] T = 8192, outliers x200
    (0, 1, 8192, 4096, 6144, 10.0),     # configs[2] T = 8192 qkv, outliers x10
    (0, 1, 2048, 4096, 28672, 10.0),    # configs[2] T = 2048 gate+up
    (0, 1, 4096, 3584, 4608, 50.0),     # configs[3] Qwen qkv, NVFP4
    (1, 1, 4096, 3584, 4608, 50.0),     #                       MXFP4
    (1, 0, 4096, 3584, 3584, 50.0),     # configs[3] Qwen o, MXFP4
    (0, 1, 4096, 3584, 37888, 50.0),    # configs[3] Qwen gate+up, NVFP4
    (1, 1, 4096, 3584, 37888, 50.0),    #                          MXFP4
]


@pytest.mark.parametrize("fmt,norm,T,K,D,mult", PREFILL_VARIANTS)
def test_prefill_launch_variants_sampled(sq, fmt, norm, T, K, D, mult):
    """BASELINE.json configs[2] / configs[3] at full size in the launch configuration bench.py times: the CTA-pair
    kernel with 192- and 256-wide tiles, a ragged last N tile, ragged T and an odd number of 128-row blocks.
    The sampled output features always include the last 64 columns (the tail of a ragged last tile) and the
    sampled rows the first / last rows of the last row block."""
    plan = sq.linear_plan(sq.make_config(fmt, norm, 1e-6, sq.LAYOUT_TILED), T, D, K)
    assert plan.startswith("pair "), plan                           # every prefill shape runs on CTA-pair tiles
    if D % 256 != 0:
        assert "bn=256" not in plan, plan                           # a ragged last N tile
    _sampled_check(sq, fmt, norm, T, K, D, config=3, mult=mult, n_rows=20, n_cols=160, seed_extra=T + D + fmt)


def test_linear_plan_names_the_variants_the_tests_cover(sq):
    """sharq_linear_plan: the decode / prefill / MoE shapes of BASELINE.json map onto the kernel variants the parity
    tests above run (split-K clusters, 128 x 256 tiles, persistent tiles, CTA pairs of both widths, multicast)."""
    cfg = sq.make_config(0, 0, 1e-6, sq.LAYOUT_TILED)
    plans = {name: sq.linear_plan(cfg, T, D, K, E) for name, (T, D, K, E) in dict(
        o_T1=(1, 4096, 4096, 0), gate_up_T128=(128, 28672, 4096, 0), down_T256=(256, 4096, 14336, 0),
        o_T4096=(4096, 4096, 4096, 0), down_T4096=(4096, 4096, 14336, 0), moe_gate_up=(40576, 1536, 2048, 128),
        moe_down=(40576, 2048, 768, 128)).items()}
    assert plans["o_T1"].startswith("tile bn=128 act_rows=16") and "splits=1 " not in plans["o_T1"], plans
    assert plans["gate_up_T128"].startswith("tile bn=256"), plans
    assert plans["o_T4096"].startswith("pair "), plans
    assert plans["down_T4096"].startswith("pair "), plans
    assert plans["moe_gate_up"].startswith("grouped-mc") and plans["moe_down"].startswith("grouped-mc"), plans
    assert sq.linear_plan(cfg, 40576, 1536, 4096, 128).startswith("grouped-pair")   # long K, > 192 rows per expert
    assert sq.linear_plan(sq.make_config(2, 0), 4096, 3584, 18944).startswith("hif4-bf16")


def test_linear_grouped_device_offsets_and_spare_capacity(sq):
    """sharq_linear_grouped reads `offsets` on the DEVICE (no host copy): a device tensor, buffers larger than the
    padded total (roundup(total, 128) + 128 E), an odd number of n-tiles (the non-multicast grouped path) and a
    capacity that is too SMALL (extra row blocks are skipped, nothing is written beyond the buffers)."""
    E = 5
    counts = [3, 0, 257, 128, 64]
    offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    pad_off = np.concatenate([[0], np.cumsum([-(-c // 128) * 128 for c in counts])])
    cap = int(-(-offsets[-1] // 128) * 128 + 128 * E)
    cfg = sq.make_config(sq.NVFP4, sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
    # 2 n-tiles (multicast clusters) / 3 (plain persistent) / long K: CTA-pair tiles on two row blocks of one expert,
    # ragged last n-tile (D = 256 with 192-wide tiles reads the next expert's weight rows, never stored)
    # ... and medium K with D % 384 == 0: 128 x 192 multicast tiles (tiles that start inside a 128-row scale atom)
    for D, K in ((256, 512), (384, 512), (256, 4096), (384, 2048), (768, 1280)):
        act = sq.alloc_act(cfg, cap, K, "cuda")
        ws, xs = [], []
        for e in range(E):
            ws.append(si.weight(D, K, 5, extra=50 + e))
            xs.append(si.activations(counts[e], K, config=5, extra=60 + e))
            if counts[e]:
                sq.prepare(cfg, to_dev(xs[e]), out=sq.act_slot(cfg, act, int(pad_off[e]), counts[e]))
        wqs = [sq.quantize_weight(cfg, to_dev(w)) for w in ws]
        wq = dict(codes=torch.cat([q["codes"] for q in wqs]), sf_sp=torch.cat([q["sf_sp"] for q in wqs]),
                  sf_dn=torch.cat([q["sf_dn"] for q in wqs]), ts_w=torch.cat([q["ts_w"] for q in wqs]), D=D, K=K)
        offs_dev = torch.from_numpy(offsets).cuda()
        assert sq.linear_plan(cfg, cap, D, K, E).startswith("grouped-pair") == (K >= 4096)   # 230 rows of capacity per expert
        assert not sq.linear_plan(cfg, 4 * 128, D, K, E).startswith("grouped-pair")
        Y = torch.full((cap, D), 7.0, dtype=torch.float32, device="cuda")
        sq.linear_grouped(cfg, offs_dev, act, wq, D, Y=Y)
        torch.cuda.synchronize()
        Yh = Y.cpu().numpy()
        for e in range(E):
            if counts[e]:
                y64 = so.linear(so.prepare(xs[e], norm=0), so.quantize_weight(ws[e]))
                assert rel_err(Yh[pad_off[e]: pad_off[e] + counts[e]], y64).max() <= TOL, f"D{D} expert {e}"
        assert (Yh[pad_off[-1]:] == 7.0).all(), "rows beyond the padded total were written"
        # capacity of 4 row blocks only (experts 0, 2 (two of its three blocks... all three), 3 need 1 + 3 + 1 + 1 = 6)
        small = dict(act, T=4 * 128)
        Y2 = torch.full((cap, D), 7.0, dtype=torch.float32, device="cuda")
        sq.linear_grouped(cfg, offs_dev, small, wq, D, Y=Y2)
        torch.cuda.synchronize()
        Y2h = Y2.cpu().numpy()
        assert (Y2h[4 * 128:] == 7.0).all(), "row blocks beyond padded_rows were computed"
        assert np.array_equal(Y2h[:3], Yh[:3])


def test_moe_config5_down_projection_sampled(sq):
    """BASELINE.json configs[4], the expert DOWN projection 768 -> 2048 (3 k-blocks, multicast clusters): the
    32768 routed rows are prepared per row into the experts' 128-row-aligned slots; three experts are checked."""
    E, K, D = 128, 768, 2048
    ids, offsets, order = si.moe_routing()
    counts = np.diff(offsets)
    cfg = sq.make_config(sq.NVFP4, sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
    pad_off = np.concatenate([[0], np.cumsum(-(-counts // 128) * 128)])
    act = sq.alloc_act(cfg, int(pad_off[-1]), K, "cuda")
    x = si.activations(int(offsets[-1]), K, config=5, extra=3)      # routed rows, already grouped by expert
    check = [int(np.argmax(counts)), int(np.argmin(counts)), 5]
    ws, wq_parts = {}, []
    for e in range(E):
        w = si.weight(D, K, 5, extra=2000 + e) if e in check else si.weight(D, K, 5, extra=3000 + e % 3)
        if e in check:
            ws[e] = w
        wq_parts.append(sq.quantize_weight(cfg, to_dev(w)))
        if counts[e]:
            sq.prepare(cfg, to_dev(x[offsets[e]: offsets[e + 1]]), out=sq.act_slot(cfg, act, int(pad_off[e]), int(counts[e])))
    wq = dict(codes=torch.cat([q["codes"] for q in wq_parts]), sf_sp=torch.cat([q["sf_sp"] for q in wq_parts]),
              sf_dn=torch.cat([q["sf_dn"] for q in wq_parts]), ts_w=torch.cat([q["ts_w"] for q in wq_parts]), D=D, K=K)
    Y = sq.linear_grouped(cfg, offsets, act, wq, D, out_dtype="fp32")
    torch.cuda.synchronize()
    Y = Y.cpu().numpy()
    for e in check:
        if counts[e] == 0:
            continue
        y64 = so.linear(so.prepare(x[offsets[e]: offsets[e + 1]], norm=0), so.quantize_weight(ws[e]))
        got = Y[pad_off[e]: pad_off[e] + counts[e]]
        assert rel_err(got, y64).max() <= TOL, f"expert {e}"


@pytest.mark.parametrize("fmt,T,K,D", [(0, 16, 1024, 200), (0, 300, 512, 328), (1, 130, 768, 136), (0, 1, 4096, 4104),
                                       (0, 512, 1024, 9480)])
def test_linear_any_multiple_of_8_columns(sq, fmt, T, K, D):
    """D % 8 == 0.  The last n-tile is ragged: W rows beyond D are zero-filled by TMA, columns beyond
    D are neither stored nor touched (sentinel columns), in the split-K, persistent and CTA-pair variants."""
    x, w, bias = si.activations(T, K, config=3, extra=D), si.weight(D, K, 3, extra=D + 1), si.beta(D, 3)
    cfg = sq.make_config(fmt, sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
    wq, act = sq.quantize_weight(cfg, to_dev(w)), sq.prepare(cfg, to_dev(x))
    big = torch.full((T, D + 24), 7.0, dtype=torch.float32, device="cuda")
    sq.linear(cfg, act, wq, bias=to_dev(bias), Y=big[:, :D])
    y16 = sq.linear(cfg, act, wq, bias=to_dev(bias), out_dtype="bf16")
    torch.cuda.synchronize()
    assert (big[:, D:] == 7.0).all(), "columns beyond D were written"
    p, q = so.prepare(x, fmt=fmt, norm=0), so.quantize_weight(w, fmt=fmt)
    assert rel_err(big[:, :D].cpu().numpy(), so.linear(p, q, bias_u16=bias)).max() <= TOL
    assert torch.equal(y16, big[:, :D].to(torch.bfloat16))


def test_outputs_are_repeatable_and_stay_inside_their_buffers(sq):
    """compute-sanitizer is closed on this GPU pool, so the races / stray writes it would look for are hunted with what
    can run here: every kernel variant 12 times on the same inputs must give bit-identical outputs (the split-K DSMEM
    exchange, the multicast grouped clusters, the CTA pairs and the lagged prepare loop all order their sums), and
    sentinel bytes around every output buffer must survive."""
    def guarded(n, dtype=torch.uint8):
        buf = torch.full((n + 512,), 0x5A if dtype == torch.uint8 else 7.0, dtype=dtype, device="cuda")
        return buf, buf[256: 256 + n]
    cases = [(1, 4096, 4096), (16, 14336, 4096), (130, 1024, 384), (256, 4096, 28672), (700, 9216, 512)]
    cfg = sq.make_config(sq.NVFP4, sq.NORM_RMS, 1e-6, sq.LAYOUT_TILED)
    for T, K, D in cases:
        x, g, w = si.activations(T, K, config=2, extra=T), si.gamma(K, 2), si.weight(D, K, 2, extra=K)
        wq = sq.quantize_weight(cfg, to_dev(w))
        xd, gd = to_dev(x), to_dev(g)
        n = sq.act_sizes(cfg, T, K)
        first = None
        for rep in range(12):
            bufs = {k: guarded(sz) for k, sz in zip(("sp_codes", "sp_sf", "sp_meta", "dn_codes", "dn_sf"), n[:5])}
            rs_full, rs = guarded(T, torch.float32)
            act = dict({k: v[1] for k, v in bufs.items()}, row_scale=rs, T=T, K=K)
            sq.capi.sharq_act_init(__import__("ctypes").byref(cfg), T, K, act["sp_sf"].data_ptr(), act["sp_meta"].data_ptr(),
                                   act["dn_sf"].data_ptr(), torch.cuda.current_stream().cuda_stream)
            sq.prepare(cfg, xd, gd, out=act)
            y_full, y = guarded(T * D, torch.float32)
            Y = y.view(T, D)
            sq.linear(cfg, act, wq, Y=Y)
            torch.cuda.synchronize()
            for k, (full, view) in bufs.items():
                assert (full[:256] == 0x5A).all() and (full[256 + view.numel():] == 0x5A).all(), f"{k} T{T} K{K}"
            assert (rs_full[:256] == 7.0).all() and (rs_full[256 + T:] == 7.0).all()
            assert (y_full[:256] == 7.0).all() and (y_full[256 + T * D:] == 7.0).all()
            snap = [act[k].clone() for k in ("sp_codes", "sp_sf", "sp_meta", "dn_codes", "dn_sf")] + [Y.clone()]
            if first is None:
                first = snap
            else:
                for a, b in zip(first, snap):
                    assert torch.equal(a, b), f"run {rep} differs (T{T} K{K} D{D})"


@pytest.mark.parametrize("fmt,norm,T,K,D", [(0, 1, 1, 4096, 4096), (0, 1, 8, 4096, 6144), (0, 0, 3, 14336, 4096), (0, 1, 2, 4096, 28672),
                                            (1, 1, 4, 3584, 512), (0, 1, 16, 4096, 4096), (0, 2, 2, 1024, 256)])
def test_prepare_linear_one_call(sq, fmt, norm, T, K, D):
    """sharq_prepare_linear: the chained pair (default) and, for T <= 8, the single fused launch (every
    GEMM CTA prepares the rows with extra warps); either way the activation operands and Y are bit-identical to
    sharq_prepare followed by sharq_linear, which the other tests compare with the oracle."""
    x = si.activations(T, K, config=2, outlier_mult=50.0, extra=T + K + D)
    g, b, w, bias = si.gamma(K, 2), si.beta(K, 2), si.weight(D, K, 2, extra=D), si.beta(D, 2)
    cfg = sq.make_config(fmt, norm, 1e-6, sq.LAYOUT_TILED)
    wq = sq.quantize_weight(cfg, to_dev(w))
    xd, gd, bd = to_dev(x), to_dev(g) if norm else None, to_dev(b) if norm == 2 else None
    act_ref = sq.prepare(cfg, xd, gd, bd)
    y_ref = sq.linear(cfg, act_ref, wq, bias=to_dev(bias), out_dtype="fp32")
    for rep in range(4):                                 # repeated: the fused launch re-reads what its own warps wrote
        y, act = sq.prepare_linear(cfg, xd, wq, gd, bd, bias=to_dev(bias), out_dtype="fp32", single_launch=rep != 3)
        torch.cuda.synchronize()
        for k in ("sp_codes", "sp_sf", "sp_meta", "dn_codes", "dn_sf", "row_scale"):
            assert torch.equal(act[k], act_ref[k]), f"{k} (rep {rep})"
        assert torch.equal(y, y_ref), f"Y (rep {rep})"
    p, q = so.prepare(x, fmt=fmt, norm=norm, gamma_u16=g, beta_u16=b if norm == 2 else None), so.quantize_weight(w, fmt=fmt)
    assert rel_err(y.cpu().numpy(), so.linear(p, q, bias_u16=bias)).max() <= TOL


@pytest.mark.parametrize("T,K,D", [(600, 768, 3328), (1000, 1024, 2304)])
def test_hif4_sparse_backbone_paths(sq, T, K, D):
    """HiF4 on the 2:4-sparse bf16 tensor path (tcgen05.mma.sp kind::f16 on the compressed survivors + metadata, dense
    MMAs on the residual; 224- and 192-wide CTA-pair tiles, ragged last n-tile, ragged T, odd number of row blocks):
    SharQ, sparse-only and dense-only against the oracle's fp64 products of the same dequantized operands."""
    x, g, w = si.activations(T, K, config=4, outlier_mult=50.0, extra=T), si.gamma(K, 4), si.weight(D, K, 4, extra=D)
    cfg = sq.make_config(sq.HIF4, sq.NORM_RMS, 1e-6)
    wq = sq.quantize_weight(cfg, to_dev(w))
    act = sq.prepare(cfg, to_dev(x), to_dev(g))
    p, q = so.prepare(x, fmt=so.HIF4, norm=1, gamma_u16=g), so.quantize_weight(w, so.HIF4)
    for path in (0, 1, 2):
        y = sq.linear(cfg, act, wq, out_dtype="fp32", path=path)
        torch.cuda.synchronize()
        err = rel_err(y.cpu().numpy(), path_reference(p, q, path))
        assert err.max() <= TOL, f"path {path}: {err.max():.3e} at {np.unravel_index(err.argmax(), err.shape)}"
    y16 = sq.linear(cfg, act, wq, out_dtype="bf16")
    assert torch.equal(y16, sq.linear(cfg, act, wq, out_dtype="fp32").to(torch.bfloat16))
