"""GPU parity of the Table 5 path combinations: Dense+Dense and
Sparse+Sparse through sharq_prepare_paths / sharq_linear_paths vs the oracle's prepare_paths / linear_paths.
Operand bytes bit-exact, GEMM within 1e-3 (R15)."""
import numpy as np
import pytest
import torch

import sharq_inputs as si
from oracle import sharq_oracle as so
from tests.gpu_util import host, to_dev

pytestmark = pytest.mark.gpu
TOL = 1e-3


@pytest.fixture(scope="module")
def sq():
    import __graft_entry__ as g
    g.build()
    import paper_2606_26587_b200 as pkg
    return pkg


def _canonical(sq, cfg, act, T, K):
    fmt, dense = cfg.fmt, act["path"] == sq.PATH_DENSE_DENSE
    C = (K // 16 if fmt == sq.NVFP4 else K // 32) if dense else K // 32
    out = {}
    for i in (0, 1):
        nb = K // 2 if dense else K // 4
        out[f"a{i}_codes"] = host(act[f"a{i}_codes"], T * nb).reshape(T, nb)
        if cfg.layout == sq.LAYOUT_TILED:
            out[f"a{i}_sf"] = host(sq.untile_sf(act[f"a{i}_sf"], T, C))
            out[f"a{i}_meta"] = None if dense else host(sq.untile_meta(act[f"a{i}_meta"], T, K))
        else:
            out[f"a{i}_sf"] = host(act[f"a{i}_sf"], T * C).reshape(T, C)
            out[f"a{i}_meta"] = None if dense else host(act[f"a{i}_meta"], T * K // 16).reshape(T, K // 16)
    out["ts"] = host(act["row_scale"])[:T]
    return out


@pytest.mark.parametrize("path", [3, 4])
@pytest.mark.parametrize("fmt,norm,layout,T,K", [(0, 1, 1, 16, 4096), (0, 0, 0, 37, 768), (1, 1, 1, 130, 3584),
                                                 (0, 2, 0, 5, 33792), (1, 0, 0, 9, 1024)])
def test_prepare_paths_bit_exact(sq, path, fmt, norm, layout, T, K):
    x = si.activations(T, K, config=3, outlier_mult=50.0, extra=K + T + path)
    g, b = si.gamma(K, 3), si.beta(K, 3)
    cfg = sq.make_config(fmt, norm, 1e-6, layout)
    act = sq.prepare_paths(cfg, path, to_dev(x), to_dev(g) if norm else None, to_dev(b) if norm == 2 else None)
    torch.cuda.synchronize()
    p = so.prepare_paths(x, path, fmt=fmt, norm=norm, gamma_u16=g, beta_u16=b if norm == 2 else None)
    got = _canonical(sq, cfg, act, T, K)
    for key in ("a0_sf", "a0_codes", "a0_meta", "a1_sf", "a1_codes", "a1_meta"):
        if p[key] is None:
            continue
        eq = got[key] == p[key]
        assert eq.all(), f"path {path} {key}: {np.count_nonzero(~eq)} of {eq.size} differ, first {np.argwhere(~eq)[:3].tolist()}"
    assert np.array_equal(got["ts"].view(np.uint32), p["ts"].view(np.uint32))


@pytest.mark.parametrize("path", [3, 4])
@pytest.mark.parametrize("fmt,norm,T,K,D", [(0, 1, 16, 4096, 4096), (0, 0, 300, 1024, 384), (1, 1, 130, 3584, 512),
                                            (0, 1, 1, 768, 256)])
def test_linear_paths_vs_oracle(sq, path, fmt, norm, T, K, D):
    x = si.activations(T, K, config=3, outlier_mult=50.0, extra=7 * T + K + path)
    g, w, bias = si.gamma(K, 3), si.weight(D, K, 3, extra=D), si.beta(D, 3)
    cfg = sq.make_config(fmt, norm, 1e-6, sq.LAYOUT_TILED)
    wq = sq.quantize_weight(cfg, to_dev(w))
    act = sq.prepare_paths(cfg, path, to_dev(x), to_dev(g) if norm else None)
    y32 = sq.linear_paths(cfg, act, wq, out_dtype="fp32")
    y16 = sq.linear_paths(cfg, act, wq, out_dtype="bf16")
    yb = sq.linear_paths(cfg, act, wq, bias=to_dev(bias), out_dtype="fp32")
    torch.cuda.synchronize()
    p = so.prepare_paths(x, path, fmt=fmt, norm=norm, gamma_u16=g)
    q = so.quantize_weight(w, fmt=fmt)
    y64 = so.linear_paths(p, q)
    den = np.maximum(np.abs(y64), 1e-2 * np.sqrt((y64 ** 2).mean()))
    err = np.abs(y32.cpu().numpy().astype(np.float64) - y64) / den
    assert err.max() <= TOL, f"path {path}: max rel err {err.max():.3e}"
    assert torch.equal(y16, y32.to(torch.bfloat16))
    yb64 = y64 + so.bf16_to_f32(bias).astype(np.float64)[None, :]
    denb = np.maximum(np.abs(yb64), 1e-2 * np.sqrt((yb64 ** 2).mean()))
    assert (np.abs(yb.cpu().numpy().astype(np.float64) - yb64) / denb).max() <= TOL


def test_paths_reject_what_they_do_not_cover(sq):
    cfg = sq.make_config(sq.HIF4)
    x = to_dev(si.activations(4, 256, config=3))
    with pytest.raises(sq.SharqError):
        sq.prepare_paths(cfg, 3, x)
    cfg = sq.make_config(sq.NVFP4, sq.NORM_NONE)
    with pytest.raises(sq.SharqError):
        sq.prepare_paths(cfg, 1, x)                    # paths 0-2 are sharq_prepare + sharq_linear's `path`
    act = sq.prepare(cfg, x)
    wq = sq.quantize_weight(cfg, to_dev(si.weight(128, 256, 3)))
    with pytest.raises(sq.SharqError):
        sq.linear(cfg, act, wq, path=3)
