"""Thin Python binding of libsharq.so (include/sharq.h).  Argument marshalling only: every step of
the SharQ hot path runs in the CUDA kernels behind the C ABI.  PyTorch is used here for device
memory and streams, nothing else.  There is no CPU fallback: a missing library raises.

Low level  : `capi.sharq_prepare(...)` etc. -- the raw ctypes functions, same names as the header.
Convenience: `quantize_weight`, `prepare`, `linear`, `linear_grouped` -- allocate the output tensors
             with the sizes the library reports, pass raw pointers + the current stream.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, c_char_p, c_float, c_int32, c_int64, c_size_t, c_void_p

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("SHARQ_LIB") or os.path.join(_HERE, "libsharq.so")   # SHARQ_LIB: another build of the same ABI

OK, EINVAL, ESHAPE, EWORKSPACE, EARCH, ECUDA = range(6)
NVFP4, MXFP4, HIF4 = 0, 1, 2
MASK_PAIR48, MASK_24 = 0, 1
NORM_NONE, NORM_RMS, NORM_LAYER = 0, 1, 2
LAYOUT_CANONICAL, LAYOUT_TILED = 0, 1
PATH_SHARQ, PATH_SPARSE_ONLY, PATH_DENSE_ONLY, PATH_DENSE_DENSE, PATH_SPARSE_SPARSE = 0, 1, 2, 3, 4
_STATUS = {0: "SHARQ_OK", 1: "SHARQ_EINVAL", 2: "SHARQ_ESHAPE", 3: "SHARQ_EWORKSPACE", 4: "SHARQ_EARCH",
           5: "SHARQ_ECUDA"}


class SharqError(RuntimeError):
    def __init__(self, status: int, where: str):
        super().__init__(f"{where} returned {_STATUS.get(status, status)}")
        self.status = status


class Config(ctypes.Structure):
    _fields_ = [("fmt", c_int32), ("mask", c_int32), ("norm", c_int32), ("eps", c_float), ("layout", c_int32)]


def make_config(fmt=NVFP4, norm=NORM_RMS, eps=1e-6, layout=LAYOUT_TILED, mask=None) -> Config:
    if mask is None:
        mask = MASK_24 if fmt == HIF4 else MASK_PAIR48
    if fmt == HIF4:
        layout = LAYOUT_CANONICAL
    return Config(fmt, mask, norm, eps, layout)


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no fallback path)")
    lib = ctypes.CDLL(LIB_PATH)
    P, SZ = c_void_p, POINTER(c_size_t)
    CFG = POINTER(Config)
    lib.sharq_version.restype = c_char_p
    lib.sharq_version.argtypes = []
    lib.sharq_weight_sizes.argtypes = [CFG, c_int64, c_int64, SZ, SZ, SZ, SZ]
    lib.sharq_act_sizes.argtypes = [CFG, c_int64, c_int64, SZ, SZ, SZ, SZ, SZ, SZ]
    lib.sharq_linear_workspace.argtypes = [CFG, c_int64, c_int64, c_int64, c_int32, SZ]
    lib.sharq_quantize_weight.argtypes = [CFG, P, c_int64, c_int64, c_int64, P, P, P, P, P, c_size_t, P]
    lib.sharq_prepare.argtypes = [CFG, P, c_int64, c_int64, c_int64, P, P, P, P, P, P, P, P, P, P]
    lib.sharq_prepare_add.argtypes = [CFG, P, P, c_int64, c_int64, c_int64, c_int64, P, c_int64, P, P, P, P, P, P, P, P, P, P]
    lib.sharq_prepare_swiglu.argtypes = [CFG, P, P, c_int64, c_int64, c_int64, c_int64, P, P, P, P, P, P, P, P, P, P]
    lib.sharq_linear.argtypes = [CFG, c_int64, c_int64, c_int64, P, P, P, P, P, P, P, P, P, P, P, P, c_int64,
                                 c_int32, c_int32, P, c_size_t, P]
    lib.sharq_prepare_linear.argtypes = [CFG, P, c_int64, c_int64, c_int64, P, P, P, P, P, P, P, P, P, c_int64, P, P, P, P, P,
                                         P, c_int64, c_int32, c_int32, P, c_size_t, P]
    lib.sharq_linear_hif4_static.argtypes = [CFG, c_int64, c_int64, c_int64, P, P, P, P, P, P, P, P, P, P, P, P, c_int64,
                                             c_int32, c_int32, P]
    lib.sharq_linear_grouped.argtypes = [CFG, c_int32, P, c_int64, c_int64, c_int64, P, P, P, P, P, P, P, P,
                                         P, P, P, c_int64, c_int32, P, c_size_t, P]
    lib.sharq_act_init.argtypes = [CFG, c_int64, c_int64, P, P, P, P]
    lib.sharq_act_sizes_paths.argtypes = [CFG, c_int32, c_int64, c_int64, SZ, SZ, SZ, SZ]
    lib.sharq_prepare_paths.argtypes = [CFG, c_int32, P, c_int64, c_int64, c_int64, P, P, P, P, P, P, P, P, P, P, P]
    lib.sharq_linear_paths.argtypes = [CFG, c_int32, c_int64, c_int64, c_int64, P, P, P, P, P, P, P, P, P, P, P, P, P,
                                       c_int64, c_int32, P]
    lib.sharq_linear_plan.argtypes = [CFG, c_int64, c_int64, c_int64, c_int32, ctypes.c_char_p, c_size_t]
    lib.sharq_untile_sf.argtypes = [P, c_int64, c_int64, P, P]
    lib.sharq_untile_meta.argtypes = [P, c_int64, c_int64, P, P]
    lib.sharq_mma_peak_launch.argtypes = [c_int32, c_int32, P]           # include/sharq_diag.h
    for name in EXPORTS[1:]:
        getattr(lib, name).restype = c_int32
    return lib


# every symbol include/sharq.h declares, then include/sharq_diag.h's
EXPORTS = ("sharq_version", "sharq_weight_sizes", "sharq_act_sizes", "sharq_linear_workspace",
           "sharq_quantize_weight", "sharq_prepare", "sharq_prepare_add", "sharq_prepare_swiglu", "sharq_prepare_linear", "sharq_linear", "sharq_linear_grouped",
           "sharq_linear_hif4_static", "sharq_act_init", "sharq_linear_plan", "sharq_untile_sf", "sharq_untile_meta", "sharq_act_sizes_paths",
           "sharq_prepare_paths", "sharq_linear_paths", "sharq_mma_peak_launch")
capi = _load()


def version() -> str:
    return capi.sharq_version().decode()


def _check(status: int, where: str):
    if status != OK:
        raise SharqError(status, where)


def _ptr(t):
    if t is None:
        return None
    if isinstance(t, int):
        return t
    return t.data_ptr()


def _stream():
    import torch
    return torch.cuda.current_stream().cuda_stream


def weight_sizes(cfg: Config, D: int, K: int):
    s = [c_size_t() for _ in range(4)]
    _check(capi.sharq_weight_sizes(ctypes.byref(cfg), D, K, *[ctypes.byref(v) for v in s]), "sharq_weight_sizes")
    return tuple(v.value for v in s)


def act_sizes(cfg: Config, T: int, K: int):
    s = [c_size_t() for _ in range(6)]
    _check(capi.sharq_act_sizes(ctypes.byref(cfg), T, K, *[ctypes.byref(v) for v in s]), "sharq_act_sizes")
    return tuple(v.value for v in s)


def linear_workspace(cfg: Config, T: int, D: int, K: int, E: int = 0) -> int:
    s = c_size_t()
    _check(capi.sharq_linear_workspace(ctypes.byref(cfg), T, D, K, E, ctypes.byref(s)), "sharq_linear_workspace")
    return s.value


def mma_peak_launch(mode: int, iters: int):
    """Diagnostics: launch the tensor-pipe issue-rate probe on the current stream (see sharq.h)."""
    _check(capi.sharq_mma_peak_launch(mode, iters, _stream()), "sharq_mma_peak_launch")


def linear_plan(cfg: Config, T: int, D: int, K: int, E: int = 0) -> str:
    """Which kernel variant sharq_linear (E == 0) / sharq_linear_grouped (E > 0, T = padded rows) launches."""
    buf = ctypes.create_string_buffer(256)
    _check(capi.sharq_linear_plan(ctypes.byref(cfg), T, D, K, E, buf, 256), "sharq_linear_plan")
    return buf.value.decode()


def untile_sf(tiled, R: int, C: int):
    """TILED scale factors (device uint8) -> canonical [R, C] device tensor, through the C ABI."""
    import torch
    out = torch.empty((R, C), dtype=torch.uint8, device=tiled.device)
    _check(capi.sharq_untile_sf(_ptr(tiled), R, C, _ptr(out), _stream()), "sharq_untile_sf")
    return out


def untile_meta(tiled, R: int, K: int):
    import torch
    out = torch.empty((R, K // 16), dtype=torch.uint8, device=tiled.device)
    _check(capi.sharq_untile_meta(_ptr(tiled), R, K, _ptr(out), _stream()), "sharq_untile_meta")
    return out


def _bytes(n, device):
    import torch
    return torch.empty(max(int(n), 16), dtype=torch.uint8, device=device)


def quantize_weight(cfg: Config, W):
    """W: torch bf16 [D, K] on cuda.  Returns dict(codes, sf_sp, sf_dn, ts_w, D, K) of device tensors."""
    import torch
    D, K = W.shape
    n_codes, n_sp, n_dn, n_ws = weight_sizes(cfg, D, K)
    dev = W.device
    out = dict(codes=_bytes(n_codes, dev), sf_sp=_bytes(n_sp, dev), sf_dn=_bytes(n_dn, dev),
               ts_w=torch.empty(1, dtype=torch.float32, device=dev), D=D, K=K)
    ws = _bytes(n_ws, dev)
    _check(capi.sharq_quantize_weight(ctypes.byref(cfg), _ptr(W), D, K, W.stride(0), _ptr(out["codes"]),
                                      _ptr(out["sf_sp"]), _ptr(out["sf_dn"]), _ptr(out["ts_w"]), _ptr(ws), n_ws,
                                      _stream()), "sharq_quantize_weight")
    return out


def alloc_act(cfg: Config, T: int, K: int, device):
    import torch
    n = act_sizes(cfg, T, K)
    out = dict(sp_codes=_bytes(n[0], device), sp_sf=_bytes(n[1], device), sp_meta=_bytes(n[2], device),
               dn_codes=_bytes(n[3], device), dn_sf=_bytes(n[4], device),
               row_scale=torch.empty(max(T, 1), dtype=torch.float32, device=device), T=T, K=K)
    if T > 0:   # pad rows of the TILED scale / metadata tiles must hold valid operands (sharq.h "Output layouts")
        _check(capi.sharq_act_init(ctypes.byref(cfg), T, K, _ptr(out["sp_sf"]), _ptr(out["sp_meta"]), _ptr(out["dn_sf"]),
                                   _stream()), "sharq_act_init")
    return out


def prepare(cfg: Config, x, gamma=None, beta=None, x_tensor_scale=None, out=None):
    """x: torch bf16 [T, K] on cuda; gamma/beta bf16 [K]; x_tensor_scale: 1-element fp32 tensor or None."""
    T, K = x.shape
    if out is None:
        out = alloc_act(cfg, T, K, x.device)
    _check(capi.sharq_prepare(ctypes.byref(cfg), _ptr(x), T, K, x.stride(0), _ptr(gamma), _ptr(beta),
                              _ptr(x_tensor_scale), _ptr(out["sp_codes"]), _ptr(out["sp_sf"]), _ptr(out["sp_meta"]),
                              _ptr(out["dn_codes"]), _ptr(out["dn_sf"]), _ptr(out["row_scale"]), _stream()),
           "sharq_prepare")
    return out


def prepare_add(cfg: Config, x, residual, gamma=None, beta=None, x_tensor_scale=None, out=None, sum_out=None):
    """sharq_prepare_add: h = bf16(x + residual) written to sum_out (default: in place over `residual`), then the
    preparation path on h.  Returns (act, sum_out)."""
    T, K = x.shape
    if out is None:
        out = alloc_act(cfg, T, K, x.device)
    if sum_out is None:
        sum_out = residual
    _check(capi.sharq_prepare_add(ctypes.byref(cfg), _ptr(x), _ptr(residual), T, K, x.stride(0), residual.stride(0),
                                  _ptr(sum_out), sum_out.stride(0), _ptr(gamma), _ptr(beta), _ptr(x_tensor_scale),
                                  _ptr(out["sp_codes"]), _ptr(out["sp_sf"]), _ptr(out["sp_meta"]), _ptr(out["dn_codes"]),
                                  _ptr(out["dn_sf"]), _ptr(out["row_scale"]), _stream()), "sharq_prepare_add")
    return out, sum_out


def prepare_paths(cfg: Config, path: int, x, gamma=None, beta=None, x_tensor_scale=None):
    """Table 5 combination (PATH_DENSE_DENSE / PATH_SPARSE_SPARSE): returns dict(a0_codes, a0_sf, a0_meta, a1_*,
    row_scale, T, K, path)."""
    import torch
    T, K = x.shape
    s = [c_size_t() for _ in range(4)]
    _check(capi.sharq_act_sizes_paths(ctypes.byref(cfg), path, T, K, *[ctypes.byref(v) for v in s]), "sharq_act_sizes_paths")
    n_codes, n_sf, n_meta, _ = (v.value for v in s)
    dev = x.device
    out = dict(T=T, K=K, path=path, row_scale=torch.empty(max(T, 1), dtype=torch.float32, device=dev))
    for i in (0, 1):
        out[f"a{i}_codes"] = _bytes(n_codes, dev)
        out[f"a{i}_sf"] = torch.zeros(max(n_sf, 16), dtype=torch.uint8, device=dev)            # pad rows: zero scales
        out[f"a{i}_meta"] = torch.full((max(n_meta, 16),), 0x44, dtype=torch.uint8, device=dev) if n_meta else None
    _check(capi.sharq_prepare_paths(ctypes.byref(cfg), path, _ptr(x), T, K, x.stride(0), _ptr(gamma), _ptr(beta),
                                    _ptr(x_tensor_scale), _ptr(out["a0_codes"]), _ptr(out["a0_sf"]), _ptr(out["a0_meta"]),
                                    _ptr(out["a1_codes"]), _ptr(out["a1_sf"]), _ptr(out["a1_meta"]), _ptr(out["row_scale"]),
                                    _stream()), "sharq_prepare_paths")
    return out


def linear_paths(cfg: Config, act: dict, wq: dict, bias=None, out_dtype="bf16", Y=None):
    import torch
    T, K, D = act["T"], act["K"], wq["D"]
    if Y is None:
        Y = torch.empty((T, D), dtype=torch.bfloat16 if out_dtype == "bf16" else torch.float32, device=act["a0_codes"].device)
    _check(capi.sharq_linear_paths(ctypes.byref(cfg), act["path"], T, D, K, _ptr(act["a0_codes"]), _ptr(act["a0_sf"]),
                                   _ptr(act["a0_meta"]), _ptr(act["a1_codes"]), _ptr(act["a1_sf"]), _ptr(act["a1_meta"]),
                                   _ptr(act["row_scale"]), _ptr(wq["codes"]), _ptr(wq["sf_sp"]), _ptr(wq["sf_dn"]),
                                   _ptr(wq["ts_w"]), _ptr(bias), _ptr(Y), Y.stride(0), 0 if Y.dtype == torch.bfloat16 else 1,
                                   _stream()), "sharq_linear_paths")
    return Y


def prepare_swiglu(cfg: Config, gate, up, gamma=None, beta=None, x_tensor_scale=None, out=None):
    """sharq_prepare_swiglu: the preparation path on h = bf16(silu(gate) * up); gate / up may be the two column halves
    of one [T, 2K] tensor."""
    T, K = gate.shape
    if out is None:
        out = alloc_act(cfg, T, K, gate.device)
    _check(capi.sharq_prepare_swiglu(ctypes.byref(cfg), _ptr(gate), _ptr(up), T, K, gate.stride(0), up.stride(0),
                                     _ptr(gamma), _ptr(beta), _ptr(x_tensor_scale), _ptr(out["sp_codes"]), _ptr(out["sp_sf"]),
                                     _ptr(out["sp_meta"]), _ptr(out["dn_codes"]), _ptr(out["dn_sf"]), _ptr(out["row_scale"]),
                                     _stream()), "sharq_prepare_swiglu")
    return out


def act_slot(cfg: Config, act: dict, row0: int, T: int) -> dict:
    """View of rows [row0, row0+T) of a TILED activation set as raw device pointers (row0 % 128 == 0):
    lets `prepare(..., out=...)` fill one expert's 128-row-aligned slot (sharq_linear_grouped, sharq.h)."""
    assert row0 % 128 == 0 and cfg.fmt != HIF4
    K = act["K"]
    c_dn = K // 16 if cfg.fmt == NVFP4 else K // 32
    return dict(sp_codes=act["sp_codes"].data_ptr() + row0 * (K // 4), sp_sf=act["sp_sf"].data_ptr() + row0 * (K // 32),
                sp_meta=act["sp_meta"].data_ptr() + row0 * (K // 16), dn_codes=act["dn_codes"].data_ptr() + row0 * (K // 2),
                dn_sf=act["dn_sf"].data_ptr() + row0 * c_dn, row_scale=act["row_scale"].data_ptr() + row0 * 4, T=T, K=K)


def linear(cfg: Config, act: dict, wq: dict, bias=None, out_dtype="bf16", path=PATH_SHARQ, Y=None, workspace=None):
    import torch
    T, K, D = act["T"], act["K"], wq["D"]
    dev = act["sp_codes"].device
    if Y is None:
        Y = torch.empty((T, D), dtype=torch.bfloat16 if out_dtype == "bf16" else torch.float32, device=dev)
    n_ws = linear_workspace(cfg, T, D, K)
    if workspace is None and n_ws:
        workspace = _bytes(n_ws, dev)
    _check(capi.sharq_linear(ctypes.byref(cfg), T, D, K, _ptr(act["sp_codes"]), _ptr(act["sp_sf"]),
                             _ptr(act["sp_meta"]), _ptr(act["dn_codes"]), _ptr(act["dn_sf"]), _ptr(act["row_scale"]),
                             _ptr(wq["codes"]), _ptr(wq["sf_sp"]), _ptr(wq["sf_dn"]), _ptr(wq["ts_w"]), _ptr(bias),
                             _ptr(Y), Y.stride(0), 0 if Y.dtype == torch.bfloat16 else 1, path, _ptr(workspace), n_ws,
                             _stream()), "sharq_linear")
    return Y


def prepare_linear(cfg: Config, x, wq: dict, gamma=None, beta=None, x_tensor_scale=None, bias=None, out_dtype="bf16",
                   act=None, Y=None, single_launch=False):
    """sharq_prepare_linear: prepare + linear as one call; single_launch=True asks for the fused launch (T <= 8, see
    sharq.h: measured slower than the chained pair).  Returns (Y, act)."""
    import torch
    T, K = x.shape
    D = wq["D"]
    if act is None:
        act = alloc_act(cfg, T, K, x.device)
    if Y is None:
        Y = torch.empty((T, D), dtype=torch.bfloat16 if out_dtype == "bf16" else torch.float32, device=x.device)
    _check(capi.sharq_prepare_linear(ctypes.byref(cfg), _ptr(x), T, K, x.stride(0), _ptr(gamma), _ptr(beta),
                                     _ptr(x_tensor_scale), _ptr(act["sp_codes"]), _ptr(act["sp_sf"]), _ptr(act["sp_meta"]),
                                     _ptr(act["dn_codes"]), _ptr(act["dn_sf"]), _ptr(act["row_scale"]), D, _ptr(wq["codes"]),
                                     _ptr(wq["sf_sp"]), _ptr(wq["sf_dn"]), _ptr(wq["ts_w"]), _ptr(bias), _ptr(Y), Y.stride(0),
                                     0 if Y.dtype == torch.bfloat16 else 1, 1 if single_launch else 0, None, 0, _stream()),
           "sharq_prepare_linear")
    return Y, act


STATIC_SCRATCH_BYTES = 8 * 1024 * 1024 + 256      # SHARQ_STATIC_SCRATCH_BYTES of sharq.h


def linear_hif4_static(cfg: Config, act: dict, wq: dict, bias=None, out_dtype="bf16", path=PATH_SHARQ, Y=None):
    """sharq_linear_hif4_static: HiF4 linear with the library's own static scratch (no workspace, no allocation in the
    call; Y may be passed in).  Raises SharqError(EWORKSPACE) beyond the limit stated in sharq.h."""
    import torch
    T, K, D = act["T"], act["K"], wq["D"]
    if Y is None:
        Y = torch.empty((T, D), dtype=torch.bfloat16 if out_dtype == "bf16" else torch.float32, device=act["sp_codes"].device)
    _check(capi.sharq_linear_hif4_static(ctypes.byref(cfg), T, D, K, _ptr(act["sp_codes"]), _ptr(act["sp_sf"]),
                                         _ptr(act["sp_meta"]), _ptr(act["dn_codes"]), _ptr(act["dn_sf"]), _ptr(act["row_scale"]),
                                         _ptr(wq["codes"]), _ptr(wq["sf_sp"]), _ptr(wq["sf_dn"]), _ptr(wq["ts_w"]), _ptr(bias),
                                         _ptr(Y), Y.stride(0), 0 if Y.dtype == torch.bfloat16 else 1, path, _stream()),
           "sharq_linear_hif4_static")
    return Y


def linear_grouped(cfg: Config, offsets, act: dict, wq: dict, D: int, out_dtype="bf16", Y=None, workspace=None):
    """offsets: DEVICE int32 tensor [E+1] (a host sequence is uploaded first); act tensors hold the 128-row-padded
    expert slots (sharq.h), act["T"] = their row capacity (a multiple of 128)."""
    import torch
    K = act["K"]
    dev = act["sp_codes"].device
    if not isinstance(offsets, torch.Tensor):
        offsets = torch.tensor([int(o) for o in offsets], dtype=torch.int32, device=dev)
    E = offsets.numel() - 1
    padded = act["T"] // 128 * 128
    if Y is None:
        Y = torch.zeros((max(padded, 1), D), dtype=torch.bfloat16 if out_dtype == "bf16" else torch.float32, device=dev)
    _check(capi.sharq_linear_grouped(ctypes.byref(cfg), E, _ptr(offsets), padded, D, K, _ptr(act["sp_codes"]),
                                     _ptr(act["sp_sf"]), _ptr(act["sp_meta"]), _ptr(act["dn_codes"]), _ptr(act["dn_sf"]),
                                     _ptr(act["row_scale"]), _ptr(wq["codes"]), _ptr(wq["sf_sp"]), _ptr(wq["sf_dn"]),
                                     _ptr(wq["ts_w"]), _ptr(Y), Y.stride(0), 0 if Y.dtype == torch.bfloat16 else 1,
                                     _ptr(workspace), 0, _stream()), "sharq_linear_grouped")
    return Y
