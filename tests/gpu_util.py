"""Helpers of the GPU parity tests: upload bf16 bit patterns, and the TILED <-> canonical index
maps restated from include/sharq.h in numpy (pure index permutations, no arithmetic of the method)."""
import numpy as np
import torch


def to_dev(u16: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(u16).view(np.int16)).cuda().view(torch.bfloat16)


def host(t: torch.Tensor, nbytes=None) -> np.ndarray:
    a = t.detach().cpu().numpy()
    return a if nbytes is None else a[:nbytes]


def untile_sf(buf: np.ndarray, R: int, C: int) -> np.ndarray:
    """TILED scale-factor bytes -> canonical [R, C] (sharq.h: 512-byte atoms of 128 rows x 4 columns)."""
    r, c = np.meshgrid(np.arange(R), np.arange(C), indexing="ij")
    off = ((r // 128) * (C // 4) + c // 4) * 512 + (r % 32) * 16 + ((r % 128) // 32) * 4 + (c % 4)
    return buf[off]


def untile_meta(buf: np.ndarray, R: int, K: int) -> np.ndarray:
    """TILED metadata bytes -> canonical [R, K/16] (2048-byte tiles of 128 rows x 16 bytes)."""
    r, b = np.meshgrid(np.arange(R), np.arange(K // 16), indexing="ij")
    off = ((r // 128) * (K // 256) + b // 16) * 2048 + (r % 128) * 16 + (b % 16)
    return buf[off]


def act_to_canonical(sq, cfg, act, T, K):
    """Device outputs of sharq_prepare -> dict of canonical numpy arrays comparable with the oracle's."""
    fmt = cfg.fmt
    out = dict(sp_codes=host(act["sp_codes"], T * K // 4).reshape(T, K // 4),
               dn_codes=host(act["dn_codes"], T * K // 2).reshape(T, K // 2),
               ts=host(act["row_scale"])[:T])
    if fmt == sq.HIF4:
        out["sp_sf"] = host(act["sp_sf"], T * K // 16).view(np.uint32).reshape(T, K // 64)
        out["dn_sf"] = host(act["dn_sf"], T * K // 16).view(np.uint32).reshape(T, K // 64)
        out["sp_meta"] = host(act["sp_meta"], T * K // 8).reshape(T, K // 8)
        return out
    Cd = K // 16 if fmt == sq.NVFP4 else K // 32
    if cfg.mask == sq.MASK_24:                              # element-wise 2:4 on E2M1: canonical only, K/8 metadata bytes
        out["sp_sf"] = host(act["sp_sf"], T * K // 32).reshape(T, K // 32)
        out["dn_sf"] = host(act["dn_sf"], T * Cd).reshape(T, Cd)
        out["sp_meta"] = host(act["sp_meta"], T * K // 8).reshape(T, K // 8)
    elif cfg.layout == sq.LAYOUT_TILED:
        # through the C ABI's own helpers (sharq_untile_sf / sharq_untile_meta) AND the numpy restatement of the
        # header's formulas: the two must agree, so neither the kernel's tiling nor the helper can drift alone
        out["sp_sf"] = host(sq.untile_sf(act["sp_sf"], T, K // 32))
        out["dn_sf"] = host(sq.untile_sf(act["dn_sf"], T, Cd))
        out["sp_meta"] = host(sq.untile_meta(act["sp_meta"], T, K))
        assert np.array_equal(out["sp_sf"], untile_sf(host(act["sp_sf"]), T, K // 32))
        assert np.array_equal(out["dn_sf"], untile_sf(host(act["dn_sf"]), T, Cd))
        assert np.array_equal(out["sp_meta"], untile_meta(host(act["sp_meta"]), T, K))
    else:
        out["sp_sf"] = host(act["sp_sf"], T * K // 32).reshape(T, K // 32)
        out["dn_sf"] = host(act["dn_sf"], T * Cd).reshape(T, Cd)
        out["sp_meta"] = host(act["sp_meta"], T * K // 16).reshape(T, K // 16)
    return out


def weight_to_canonical(sq, cfg, wq, D, K):
    out = dict(codes=host(wq["codes"], D * K // 2).reshape(D, K // 2), ts_w=float(host(wq["ts_w"])[0]))
    if cfg.fmt == sq.HIF4:
        out["sf_sp"] = host(wq["sf_sp"], D * K // 16).view(np.uint32).reshape(D, K // 64)
        out["w_bf16"] = host(wq["sf_dn"], D * K * 2).view(np.uint16).reshape(D, K)      # HiF4 dense view: exact bf16 values
        return out
    Cd = K // 16 if cfg.fmt == sq.NVFP4 else K // 32
    if cfg.layout == sq.LAYOUT_TILED:
        out["sf_sp"] = host(sq.untile_sf(wq["sf_sp"], D, K // 32))
        out["sf_dn"] = host(sq.untile_sf(wq["sf_dn"], D, Cd))
        assert np.array_equal(out["sf_sp"], untile_sf(host(wq["sf_sp"]), D, K // 32))
        assert np.array_equal(out["sf_dn"], untile_sf(host(wq["sf_dn"]), D, Cd))
    else:
        out["sf_sp"] = host(wq["sf_sp"], D * K // 32).reshape(D, K // 32)
        out["sf_dn"] = host(wq["sf_dn"], D * Cd).reshape(D, Cd)
    return out
