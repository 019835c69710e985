"""HiF4 part of the SharQ CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

HiFloat4 as the paper defines it (Appendix A.2): a unit is 64 S1P2 elements plus 32
bits of three-level scale metadata (E6M2, 8x E1, 16x E1); conversion from BF16 is Algorithm 1
(P:496-528), followed here line by line.  Readings R9-R12: round-half-to-even
everywhere (P:492-494 allows either); (1/7)_BF16 = 0.142578125; the reciprocal is the 4-entry
table bf16(1/1.M) * 2^-E; the sparse backbone runs Alg. 1 on 64 LOGICAL positions of
M (.) X; metadata word = E6M2 | E1_8 << 8 | E1_16 << 16.
"""
from __future__ import annotations

import numpy as np

F32 = np.float32
U8 = np.uint8
U16 = np.uint16
U32 = np.uint32

ONE_SEVENTH_BF16 = F32(0.142578125)                     # (1/7) rounded to bf16
REC_LUT = np.array([1.0, 0.80078125, 0.66796875, 0.5703125], dtype=F32)   # bf16(1/1.M)


def _bf16_to_f32(u16):
    return (np.asarray(u16, dtype=U16).astype(U32) << U32(16)).view(F32)


def _f32_to_bf16(x):
    u = np.ascontiguousarray(x, dtype=F32).view(U32)
    return ((u + U32(0x7FFF) + ((u >> U32(16)) & U32(1))) >> U32(16)).astype(U16)


def _round_bf16(x):
    return _bf16_to_f32(_f32_to_bf16(x))


def e6m2_encode(sf: np.ndarray) -> np.ndarray:
    """Positive bf16-valued fp32 -> E6M2 code eeeeee_mm (bias 48, hidden 1, Table 7
    P:451-459): RNE to 2 mantissa bits, clamped to [2^-48, 2^15 * 1.5]; sf == 0 -> code 0."""
    sf = np.asarray(sf, dtype=F32).astype(np.float64)
    m, e = np.frexp(sf)                                   # sf = m * 2^e, m in [0.5, 1)
    E = e - 1
    q = np.rint(np.ldexp(sf, 2 - E)).astype(np.int64)     # (1.M) * 4 rounded, in [4, 8]
    carry = q == 8
    E = np.where(carry, E + 1, E)
    q = np.where(carry, 4, q)
    code = ((E + 48) << 2) | (q - 4)
    code = np.where(sf < 2.0 ** -48, 0, code)             # below the minimum (incl. 0)
    code = np.where(sf > 1.5 * 2.0 ** 15, 0xFE, code)     # above the maximum
    code = np.where((E + 48 > 63), 0xFE, code)
    code = np.where((E + 48 < 0), 0, code)
    return code.astype(U8)


def e6m2_decode(code: np.ndarray) -> np.ndarray:
    """Eq. 14: X = 2^E * 1.M."""
    c = np.asarray(code, dtype=U8).astype(np.int64)
    return np.ldexp(1.0 + (c & 3) / 4.0, (c >> 2) - 48).astype(F32)


def e6m2_reciprocal(code: np.ndarray) -> np.ndarray:
    """E6M2_REC_to_BF16: table of bf16(1/1.M) and exponent negation."""
    c = np.asarray(code, dtype=U8).astype(np.int64)
    return np.ldexp(REC_LUT[c & 3].astype(np.float64), -((c >> 2) - 48)).astype(F32)


def s1p2_encode(v: np.ndarray) -> np.ndarray:
    """fp32 -> S1P2 code (bit3 sign, 3 magnitude bits in units of 0.25, Table 7): RNE to a
    multiple of 0.25, saturating at 1.75; sign bit = sign of v."""
    v = np.asarray(v, dtype=F32)
    mag = np.minimum(np.rint(np.abs(v).astype(np.float64) * 4.0), 7).astype(U8)
    sign = (v.view(U32) >> U32(31)).astype(U8)
    return (mag | (sign << U8(3))).astype(U8)


def s1p2_decode(code: np.ndarray) -> np.ndarray:
    code = np.asarray(code, dtype=U8)
    mag = (code & U8(7)).astype(F32) * F32(0.25)
    return np.where((code & U8(8)) != 0, -mag, mag).astype(F32)


def hif4_encode_units(V_u16: np.ndarray):
    """Algorithm 1 on every row of V_u16 [N, 64] (bf16 bits).
    Returns (s1p2 codes [N,64] u8, meta [N] u32 = E6M2 | E1_8 << 8 | E1_16 << 16)."""
    V = _bf16_to_f32(V_u16)
    N = V.shape[0]
    A = np.abs(V)
    # Stage 1: three-level tree reduction (lines 1-8)
    V16 = A.reshape(N, 16, 4).max(axis=-1)
    V8 = V16.reshape(N, 8, 2).max(axis=-1)
    Vmax = V8.max(axis=-1)
    # Stage 2: scaling metadata (lines 9-16)
    SF = _round_bf16(Vmax * ONE_SEVENTH_BF16)             # line 10, bf16 multiply
    e6m2 = e6m2_encode(SF)                                # line 11
    rec = e6m2_reciprocal(e6m2)                           # line 12
    E1_8 = (V8 * rec[:, None] >= F32(4.0))                # line 13 (product exact in fp32)
    s8 = np.where(E1_8, F32(0.5), F32(1.0))
    E1_16 = (V16 * rec[:, None] * np.repeat(s8, 2, axis=1) >= F32(2.0))   # line 14
    s16 = np.where(E1_16, F32(0.5), F32(1.0))
    # Stage 3: scale and quantise (lines 17-21); the scaled value is a BF16 (R10)
    scaled = _round_bf16(V * rec[:, None]) * np.repeat(s8, 8, axis=1) * np.repeat(s16, 4, axis=1)
    codes = s1p2_encode(scaled)
    w8 = (E1_8.astype(U32) << np.arange(8, dtype=U32)).sum(axis=1).astype(U32)
    w16 = (E1_16.astype(U32) << np.arange(16, dtype=U32)).sum(axis=1).astype(U32)
    meta = e6m2.astype(U32) | (w8 << U32(8)) | (w16 << U32(16))
    return codes, meta


def hif4_decode_units(codes: np.ndarray, meta: np.ndarray) -> np.ndarray:
    """Eq. 15 with 0-based integer division (R16): V_i = E6M2 * 2^(E1_8[i//8] +
    E1_16[i//4]) * S1P2_i.  Exact in fp32."""
    meta = np.asarray(meta, dtype=U32)
    base = e6m2_decode((meta & U32(0xFF)).astype(U8)).astype(np.float64)
    e8 = ((meta[:, None] >> (U32(8) + np.arange(8, dtype=U32))) & U32(1)).astype(np.int64)
    e16 = ((meta[:, None] >> (U32(16) + np.arange(16, dtype=U32))) & U32(1)).astype(np.int64)
    sh = np.repeat(e8, 8, axis=1) + np.repeat(e16, 4, axis=1)
    val = np.ldexp(s1p2_decode(codes).astype(np.float64), sh) * base[:, None]
    return val.astype(F32)


def _pack(codes):
    return (codes[:, 0::2] | (codes[:, 1::2] << U8(4))).astype(U8)


def _unpack(packed):
    T, n = packed.shape
    out = np.empty((T, 2 * n), dtype=U8)
    out[:, 0::2] = packed & U8(0xF)
    out[:, 1::2] = packed >> U8(4)
    return out


def prepare_hif4(x_u16, norm=1, gamma_u16=None, beta_u16=None, eps=1e-6):
    """SharQ preparation with HiF4 and the standard 2:4 pattern.
    Outputs as `sharq_oracle.prepare`, with sp_sf / dn_sf being u32 scale-metadata words
    [T, K/64] and sp_meta [T, K/8] (one nibble per 4 elements)."""
    from . import sharq_oracle as so
    x_u16 = np.asarray(x_u16, dtype=U16)
    T, K = x_u16.shape
    assert K % 256 == 0
    X = so.normalize(x_u16, norm, gamma_u16, beta_u16, eps)
    Xf = _bf16_to_f32(X)
    keep, nib = so.mask_24(X)
    sp_meta = so.pack_nibbles(nib)
    Xsp = np.where(keep, X, U16(0)).astype(U16)           # M (.) X, +0 at dropped positions
    c_all, m_sp = hif4_encode_units(Xsp.reshape(-1, 64))
    d = hif4_decode_units(c_all, m_sp).reshape(T, K)
    c_all = c_all.reshape(T, K)
    Xsp_tilde = np.where(keep, d, F32(0)).astype(F32)
    R = np.where(keep, Xf - d, Xf).astype(F32)
    sp_codes = _pack(c_all[keep].reshape(T, K // 2))
    Rb = _f32_to_bf16(R)                                  # Alg. 1 takes BF16 input
    c_dn, m_dn = hif4_encode_units(Rb.reshape(-1, 64))
    return dict(X=X, ts=np.ones(T, dtype=F32), keep=keep, sp_meta=sp_meta, sp_codes=sp_codes,
                sp_sf=m_sp.reshape(T, K // 64), Xsp_tilde=Xsp_tilde, R=R,
                dn_codes=_pack(c_dn.reshape(T, K)), dn_sf=m_dn.reshape(T, K // 64),
                fmt=2, mask=1, Gs=64, Gd=64)


def quantize_weight_hif4(w_u16):
    w_u16 = np.asarray(w_u16, dtype=U16)
    D, K = w_u16.shape
    c, m = hif4_encode_units(w_u16.reshape(-1, 64))
    m = m.reshape(D, K // 64)
    return dict(codes=_pack(c.reshape(D, K)), sf_sp=m, sf_dn=m.copy(), ts_w=F32(1.0), fmt=2)


def hif4_dequant_backbone(prep):
    from . import sharq_oracle as so
    codes, keep = so.expand_backbone(prep)
    T, K = codes.shape
    val = hif4_decode_units(codes.reshape(-1, 64), prep["sp_sf"].reshape(-1)).reshape(T, K)
    return np.where(keep, val, 0).astype(np.float64)


def hif4_dequant_residual(prep):
    codes = _unpack(prep["dn_codes"])
    T, K = codes.shape
    return hif4_decode_units(codes.reshape(-1, 64), prep["dn_sf"].reshape(-1)).reshape(T, K).astype(np.float64)


def hif4_dequant_weight(wq):
    codes = _unpack(wq["codes"])
    D, K = codes.shape
    return hif4_decode_units(codes.reshape(-1, 64), wq["sf_sp"].reshape(-1)).reshape(D, K).astype(np.float64)
