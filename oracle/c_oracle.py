"""ctypes wrapper and build step of the C oracle (oracle/sharq_oracle_c.c) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

`build()` compiles the C file with gcc (-O2, no fast-math, no FMA contraction, OpenMP) into oracle/libsharq_oracle_c.so;
the functions below only marshal numpy arrays.  No arithmetic of the method lives here.  Only tests/, __graft_entry__
and bench.py's cpu_baseline / --impl reference legs may import this module.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sharq_oracle_c.c")
LIB = os.path.join(HERE, "libsharq_oracle_c.so")
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra"]

NVFP4, MXFP4 = 0, 1
NORM_NONE, NORM_RMS, NORM_LAYER = 0, 1, 2

_lib = None


def build(force: bool = False) -> str:
    """gcc the C oracle if the library is missing or older than its source.  Returns the library path."""
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        tmp = LIB + f".tmp{os.getpid()}"
        try:
            subprocess.run(["gcc", *CFLAGS, "-o", tmp, SRC, "-lm"], check=True)
        except (OSError, subprocess.CalledProcessError):
            if force or not os.path.exists(LIB):
                raise
            return LIB              # no compiler on this box: a library shipped with the tree (copies reset mtimes)
        os.replace(tmp, LIB)
    return LIB


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.so_max_threads.restype = ctypes.c_int
        _lib.so_canonical_sum.restype = ctypes.c_float
        _lib.so_exp_neg.restype = ctypes.c_float
        _lib.so_exp_neg.argtypes = [ctypes.c_float]
    return _lib


def max_threads() -> int:
    return int(lib().so_max_threads())


def canonical_sum(row_f32, squares: bool) -> np.float32:
    t = np.ascontiguousarray(row_f32, dtype=np.float32)
    return np.float32(lib().so_canonical_sum(_p(t), ctypes.c_int64(t.size), int(bool(squares))))


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _u16(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.uint16)


def prepare(x_u16, fmt=NVFP4, norm=NORM_RMS, gamma_u16=None, beta_u16=None, eps=1e-6, x_tensor_scale=None,
            nthreads=0, want_X=True):
    """Same outputs (canonical arrays) as the numpy oracle's `prepare` for NVFP4 / MXFP4 with the pairwise 4:8 mask."""
    x = _u16(x_u16)
    T, K = x.shape
    Gd = 16 if fmt == NVFP4 else 32
    out = dict(sp_codes=np.empty((T, K // 4), np.uint8), sp_sf=np.empty((T, K // 32), np.uint8),
               sp_meta=np.empty((T, K // 16), np.uint8), dn_codes=np.empty((T, K // 2), np.uint8),
               dn_sf=np.empty((T, K // Gd), np.uint8), ts=np.empty(T, np.float32),
               X=np.empty((T, K), np.uint16) if want_X else None)
    g, b = _u16(gamma_u16), _u16(beta_u16)
    sts = None if x_tensor_scale is None else ctypes.byref(ctypes.c_float(x_tensor_scale))
    rc = lib().so_prepare(_p(x), ctypes.c_int64(T), ctypes.c_int64(K), int(fmt), int(norm), _p(g), _p(b),
                          ctypes.c_float(eps), sts, _p(out["sp_codes"]), _p(out["sp_sf"]), _p(out["sp_meta"]),
                          _p(out["dn_codes"]), _p(out["dn_sf"]), _p(out["ts"]), _p(out["X"]), int(nthreads))
    if rc < 0:
        raise ValueError(f"so_prepare rejected its arguments ({rc})")
    out.update(fmt=fmt, threads=rc, T=T, K=K)
    return out


def quantize_weight(w_u16, fmt=NVFP4, nthreads=0):
    w = _u16(w_u16)
    D, K = w.shape
    out = dict(codes=np.empty((D, K // 2), np.uint8), sf_sp=np.empty((D, K // 32), np.uint8),
               sf_dn=np.empty((D, K // (16 if fmt == NVFP4 else 32)), np.uint8))
    ts_w = ctypes.c_float(0)
    rc = lib().so_quantize_weight(_p(w), ctypes.c_int64(D), ctypes.c_int64(K), int(fmt), _p(out["codes"]),
                                  _p(out["sf_sp"]), _p(out["sf_dn"]), ctypes.byref(ts_w), int(nthreads))
    if rc < 0:
        raise ValueError(f"so_quantize_weight rejected its arguments ({rc})")
    out.update(ts_w=np.float32(ts_w.value), fmt=fmt, threads=rc, D=D, K=K)
    return out


def linear(prep, wq, rows=None, cols=None, nthreads=0):
    """fp64 [n_rows, n_cols] of Eq. 9 from the stored arrays of `prepare` and `quantize_weight`."""
    T, K, D = prep["T"], prep["K"], wq["D"]
    r = None if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    c = None if cols is None else np.ascontiguousarray(cols, dtype=np.int64)
    nr, nc = (T if r is None else len(r)), (D if c is None else len(c))
    Y = np.empty((nr, nc), np.float64)
    rc = lib().so_linear(ctypes.c_int64(T), ctypes.c_int64(K), ctypes.c_int64(D), int(prep["fmt"]),
                         _p(prep["sp_codes"]), _p(prep["sp_sf"]), _p(prep["sp_meta"]), _p(prep["dn_codes"]),
                         _p(prep["dn_sf"]), _p(prep["ts"]), _p(wq["codes"]), _p(wq["sf_sp"]), _p(wq["sf_dn"]),
                         ctypes.c_float(float(wq["ts_w"])), _p(r), ctypes.c_int64(nr), _p(c), ctypes.c_int64(nc),
                         _p(Y), int(nthreads))
    if rc < 0:
        raise ValueError(f"so_linear failed ({rc})")
    return Y


def residual_add(x_u16, r_u16):
    """h = bf16(x + r), elementwise (bf16 bit patterns)."""
    x, r = _u16(x_u16), _u16(r_u16)
    h = np.empty_like(x)
    lib().so_residual_add(_p(x), _p(r), ctypes.c_int64(x.size), _p(h))
    return h


def swiglu(gate_u16, up_u16, nthreads=0):
    """h = bf16(silu(gate) * up) with DESIGN.md R18's exp contract."""
    g, u = _u16(gate_u16), _u16(up_u16)
    h = np.empty_like(g)
    lib().so_swiglu(_p(g), _p(u), ctypes.c_int64(g.size), _p(h), int(nthreads))
    return h


def exp_neg(g: float) -> np.float32:
    return np.float32(lib().so_exp_neg(ctypes.c_float(g)))


def prepare_hif4(x_u16, norm=NORM_RMS, gamma_u16=None, beta_u16=None, eps=1e-6, nthreads=0):
    """Same stored outputs as the numpy oracle's `prepare_hif4` (2:4 mask, Algorithm 1 on backbone and residual)."""
    x = _u16(x_u16)
    T, K = x.shape
    out = dict(sp_codes=np.empty((T, K // 4), np.uint8), sp_sf=np.empty((T, K // 64), np.uint32),
               sp_meta=np.empty((T, K // 8), np.uint8), dn_codes=np.empty((T, K // 2), np.uint8),
               dn_sf=np.empty((T, K // 64), np.uint32), ts=np.ones(T, np.float32))
    g, b = _u16(gamma_u16), _u16(beta_u16)
    rc = lib().so_prepare_hif4(_p(x), ctypes.c_int64(T), ctypes.c_int64(K), int(norm), _p(g), _p(b), ctypes.c_float(eps),
                               _p(out["sp_codes"]), _p(out["sp_sf"]), _p(out["sp_meta"]), _p(out["dn_codes"]),
                               _p(out["dn_sf"]), int(nthreads))
    if rc < 0:
        raise ValueError(f"so_prepare_hif4 rejected its arguments ({rc})")
    out.update(fmt=2, threads=rc, T=T, K=K)
    return out


def quantize_weight_hif4(w_u16, nthreads=0):
    w = _u16(w_u16)
    D, K = w.shape
    out = dict(codes=np.empty((D, K // 2), np.uint8), sf_sp=np.empty((D, K // 64), np.uint32))
    rc = lib().so_quantize_weight_hif4(_p(w), ctypes.c_int64(D), ctypes.c_int64(K), _p(out["codes"]), _p(out["sf_sp"]),
                                       int(nthreads))
    if rc < 0:
        raise ValueError(f"so_quantize_weight_hif4 rejected its arguments ({rc})")
    out.update(fmt=2, threads=rc, D=D, K=K)
    return out


def linear_hif4(prep, wq, rows=None, cols=None, nthreads=0):
    T, K, D = prep["T"], prep["K"], wq["D"]
    r = None if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    c = None if cols is None else np.ascontiguousarray(cols, dtype=np.int64)
    nr, nc = (T if r is None else len(r)), (D if c is None else len(c))
    Y = np.empty((nr, nc), np.float64)
    rc = lib().so_linear_hif4(ctypes.c_int64(T), ctypes.c_int64(K), ctypes.c_int64(D), _p(prep["sp_codes"]),
                              _p(prep["sp_sf"]), _p(prep["sp_meta"]), _p(prep["dn_codes"]), _p(prep["dn_sf"]),
                              _p(wq["codes"]), _p(wq["sf_sp"]), _p(r), ctypes.c_int64(nr), _p(c), ctypes.c_int64(nc),
                              _p(Y), int(nthreads))
    if rc < 0:
        raise ValueError(f"so_linear_hif4 failed ({rc})")
    return Y
