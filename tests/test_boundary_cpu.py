"""The C-ABI library loads, exports every symbol include/sharq.h declares, and its host-only logic
(size queries, argument validation) behaves as the header says.  No compute calls (no GPU needed)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def sq():
    import __graft_entry__ as g
    g.build()
    import paper_2606_26587_b200 as pkg
    return pkg


def test_every_declared_symbol_is_exported(sq):
    declared = set()
    for h in ("sharq.h", "sharq_diag.h"):
        text = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", h)).read(), flags=re.S)   # comments mention calls too
        declared |= set(re.findall(r"\b(sharq_[a-z0-9_]+)\s*\(", text))
    assert declared == set(sq.EXPORTS)
    for name in declared:
        assert getattr(sq.capi, name) is not None
    assert sq.version().startswith("sharq-b200")


def test_sizes_follow_the_header(sq):
    cfg = sq.make_config(sq.NVFP4, layout=sq.LAYOUT_CANONICAL)
    T, K, D = 16, 4096, 6144
    assert sq.act_sizes(cfg, T, K) == (T * K // 4, T * K // 32, T * K // 16, T * K // 2, T * K // 16, T * 4)
    assert sq.weight_sizes(cfg, D, K)[:3] == (D * K // 2, D * K // 32, D * K // 16)
    cfg_t = sq.make_config(sq.NVFP4, layout=sq.LAYOUT_TILED)
    assert sq.act_sizes(cfg_t, T, K) == (T * K // 4, 128 * K // 32, 128 * K // 16, T * K // 2, 128 * K // 16, T * 4)
    # per element: 2 B in + 0.25 + 0.0625 + 0.03125 + 0.5 + 0.0625 out = 2.906 B (DESIGN.md roofline unit)
    n = sq.act_sizes(cfg, 128, 4096)
    assert (sum(n[:5]) + 2 * 128 * 4096) / (128 * 4096) == 2.90625
    cfg_m = sq.make_config(sq.MXFP4, layout=sq.LAYOUT_CANONICAL)
    assert sq.act_sizes(cfg_m, T, K)[4] == T * K // 32
    cfg_h = sq.make_config(sq.HIF4)
    assert sq.weight_sizes(cfg_h, D, K)[:3] == (D * K // 2, D * K // 16, D * K * 2)      # dense view = bf16 [D, K]
    assert sq.act_sizes(cfg_h, T, K) == (T * K // 4, T * K // 16, T * K // 8, T * K // 2, T * K // 16, T * 4)


def test_argument_validation_returns_codes_without_touching_cuda(sq):
    cfg = sq.make_config(sq.NVFP4)
    null = ctypes.c_void_p(0)
    f = sq.capi.sharq_prepare
    # K not a multiple of 256
    assert f(ctypes.byref(cfg), 16, 4, 1000, 1000, *([16] * 9), null) == sq.ESHAPE
    # T == 0 is OK and launches nothing
    assert f(ctypes.byref(cfg), 16, 0, 1024, 1024, *([16] * 9), null) == sq.OK
    # null output pointer
    assert f(ctypes.byref(cfg), 16, 4, 1024, 1024, 16, null, null, null, 16, 16, 16, 16, 16, null) == sq.EINVAL
    # misaligned pointer
    assert f(ctypes.byref(cfg), 8, 4, 1024, 1024, 16, null, null, 16, 16, 16, 16, 16, 16, null) == sq.EINVAL
    # sharq_prepare_add: (cfg, x, residual, T, K, ldx, ldr, sum_out, ldo, gamma, beta, x_ts, 6 outputs, stream)
    g = sq.capi.sharq_prepare_add
    ok_ptrs = [32] * 9                                    # gamma, beta, x_ts, sp_codes ... row_scale
    assert g(ctypes.byref(cfg), 32, 64, 0, 1024, 1024, 1024, 96, 1024, *ok_ptrs, null) == sq.OK          # T == 0
    assert g(ctypes.byref(cfg), 32, 64, 4, 1000, 1008, 1008, 96, 1008, *ok_ptrs, null) == sq.ESHAPE      # K % 256
    assert g(ctypes.byref(cfg), 32, 64, 4, 1024, 1032, 1024, 96, 1024, *ok_ptrs, null) == sq.ESHAPE      # ldx % 16
    assert g(ctypes.byref(cfg), 32, 64, 4, 33792, 33792, 33792, 96, 33792, *ok_ptrs, null) == sq.ESHAPE  # K > 32768
    assert g(ctypes.byref(cfg), 16, 64, 4, 1024, 1024, 1024, 96, 1024, *ok_ptrs, null) == sq.EINVAL      # x 16-byte aligned only
    assert g(ctypes.byref(cfg), 32, null, 4, 1024, 1024, 1024, 96, 1024, *ok_ptrs, null) == sq.EINVAL    # no residual
    assert g(ctypes.byref(cfg), 32, 64, 4, 1024, 1024, 1024, 32, 1024, *ok_ptrs, null) == sq.EINVAL      # sum_out aliases x
    # element-wise 2:4 with NVFP4 / MXFP4: accepted by sharq_prepare / sharq_act_sizes in the canonical layout
    # (metadata K/8 bytes per row), refused by everything on the GEMM side: B200 has no such FP4 MMA (R2)
    m24 = sq.Config(sq.NVFP4, sq.MASK_24, sq.NORM_NONE, 1e-6, sq.LAYOUT_CANONICAL)
    assert sq.act_sizes(m24, 16, 1024) == (16 * 256, 16 * 32, 16 * 128, 16 * 512, 16 * 64, 64)
    assert f(ctypes.byref(m24), 16, 0, 1024, 1024, *([16] * 9), null) == sq.OK
    with pytest.raises(sq.SharqError) as e:
        sq.linear_workspace(m24, 16, 128, 1024)
    assert e.value.status == sq.ESHAPE
    bad = sq.Config(sq.NVFP4, sq.MASK_24, sq.NORM_NONE, 1e-6, sq.LAYOUT_TILED)
    with pytest.raises(sq.SharqError):
        sq.act_sizes(bad, 16, 1024)
    # sharq_linear_grouped: offsets is a device pointer; E, padded_rows are validated on the host
    lg = sq.capi.sharq_linear_grouped
    ptrs9 = [16] * 10                                     # 5 activation operands, row_scale, 3 weight tensors, ts_w
    assert lg(ctypes.byref(cfg), 4, 16, 100, 128, 256, *ptrs9, 16, 128, 0, null, 0, null) == sq.ESHAPE     # padded_rows % 128
    assert lg(ctypes.byref(cfg), 2000, 16, 128, 128, 256, *ptrs9, 16, 128, 0, null, 0, null) == sq.ESHAPE  # E > 1024
    assert lg(ctypes.byref(cfg), 4, null, 128, 128, 256, *ptrs9, 16, 128, 0, null, 0, null) == sq.EINVAL   # no offsets
    assert lg(ctypes.byref(cfg), 4, 16, 0, 128, 256, *ptrs9, 16, 128, 0, null, 0, null) == sq.OK           # nothing to do
    # untile helpers: shape rules
    assert sq.capi.sharq_untile_sf(16, 4, 6, 16, null) == sq.ESHAPE
    assert sq.capi.sharq_untile_meta(16, 4, 1000, 16, null) == sq.ESHAPE
    assert sq.capi.sharq_untile_sf(16, 0, 8, 16, null) == sq.OK
    with pytest.raises(sq.SharqError):
        sq.act_sizes(cfg, 16, 1000)
    with pytest.raises(sq.SharqError):
        sq.linear_workspace(cfg, 16, 100, 1024)          # D % 8
    assert sq.linear_workspace(cfg, 16, 200, 1024) == 0  # any multiple of 8
    with pytest.raises(sq.SharqError):
        sq.linear_workspace(sq.make_config(sq.HIF4), 16, 200, 1024)      # HiF4 emulation: D % 128
