"""sharq_linear_hif4_static: the no-allocation entry point (scratch in a file-scope device array inside libsharq.so).
Collected last on purpose (pytest -x: a failure here must not hide any other test).  Passes alone in
a fresh process and after the other tests: it shares nothing with them but the library."""
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


def _case(sq, T, K, D, norm, seed):
    x, g, w = si.activations(T, K, config=4, outlier_mult=50.0, extra=seed), si.gamma(K, 4), si.weight(D, K, 4, extra=seed + 1)
    cfg = sq.make_config(sq.HIF4, norm, 1e-6)
    wq = sq.quantize_weight(cfg, to_dev(w))
    act = sq.prepare(cfg, to_dev(x), to_dev(g) if norm else None)
    return cfg, x, g, w, wq, act


def test_static_scratch_matches_the_workspace_path_on_two_calls_in_a_row(sq):
    """Two calls in a row on different problems (the second smaller, so the array still holds the first call's bytes
    beyond its own rows): each equals the existing sharq_linear (caller's workspace) bit for bit, is within the GEMM
    tolerance of the oracle, and the calls take no device memory (driver-level free bytes unchanged)."""
    cases = [(130, 768, 384, 0, 11), (16, 4096, 4096, 1, 12)]
    prepared = [_case(sq, *c) for c in cases]
    outs = [torch.empty((c[0], c[2]), dtype=torch.float32, device="cuda") for c in cases]
    refs = [sq.linear(p[0], p[5], p[4], out_dtype="fp32") for p in prepared]          # existing path, its own workspace
    for (cfg, x, g, w, wq, act), Y in zip(prepared, outs):   # warm-up: the driver loads each kernel's code lazily on its
        sq.linear_hif4_static(cfg, act, wq, Y=Y)             # first launch (128- and 256-wide GEMM variants), which takes
    for Y in outs:                                           # device memory once per process whoever launches it
        Y.zero_()                                            # (torch's own fill kernel included: outside the measured region)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for (cfg, x, g, w, wq, act), Y in zip(prepared, outs):                            # the two calls, back to back:
        sq.linear_hif4_static(cfg, act, wq, Y=Y)                                      # nothing but the C-ABI call in here
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0, "the no-allocation entry point took device memory"
    for (cfg, x, g, w, wq, act), Y, ref, c in zip(prepared, outs, refs, cases):
        assert torch.equal(Y, ref), f"static-scratch output differs from the workspace path {c}"
        p = so.prepare(x, fmt=so.HIF4, norm=c[3], gamma_u16=g if c[3] else None)
        y64 = so.linear(p, so.quantize_weight(w, so.HIF4))
        den = np.maximum(np.abs(y64), 1e-2 * np.sqrt((y64 ** 2).mean()))
        assert (np.abs(Y.cpu().numpy().astype(np.float64) - y64) / den).max() <= TOL
    # bf16 output and bias through the same entry point
    cfg, x, g, w, wq, act = prepared[1]
    bias = to_dev(si.beta(cases[1][2], 4))
    yb = sq.linear_hif4_static(cfg, act, wq, bias=bias, out_dtype="bf16")
    torch.cuda.synchronize()
    assert torch.equal(yb, sq.linear(cfg, act, wq, bias=bias, out_dtype="bf16"))


def test_static_scratch_rejects_what_does_not_fit(sq):
    """Beyond the stated maximum (roundup(T, 128) * 2K * 2 + 256 <= SHARQ_STATIC_SCRATCH_BYTES) the call returns
    SHARQ_EWORKSPACE and launches nothing; other formats are refused (they need no scratch: use sharq_linear)."""
    T, K, D = 512, 8192, 128
    assert -(-T // 128) * 128 * 2 * K * 2 + 256 > sq.STATIC_SCRATCH_BYTES
    cfg = sq.make_config(sq.HIF4, sq.NORM_NONE)
    dummy = torch.zeros(16, dtype=torch.uint8, device="cuda")
    act = dict(sp_codes=dummy, sp_sf=dummy, sp_meta=dummy, dn_codes=dummy, dn_sf=dummy,
               row_scale=torch.ones(T, device="cuda"), T=T, K=K)
    wq = dict(codes=dummy, sf_sp=dummy, sf_dn=dummy, ts_w=torch.ones(1, device="cuda"), D=D, K=K)
    Y = torch.full((T, D), 7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(sq.SharqError) as e:
        sq.linear_hif4_static(cfg, act, wq, Y=Y)
    assert e.value.status == sq.EWORKSPACE
    torch.cuda.synchronize()
    assert (Y == 7.0).all()
    with pytest.raises(sq.SharqError) as e:
        sq.linear_hif4_static(sq.make_config(sq.NVFP4, sq.NORM_NONE), dict(act, T=16), wq, Y=Y[:16])
    assert e.value.status == sq.EINVAL
    # the largest shapes the header promises do fit
    for t, k in ((128, 16384), (256, 8192), (512, 4096)):
        assert -(-t // 128) * 128 * 2 * k * 2 + 256 <= sq.STATIC_SCRATCH_BYTES
