"""SharQ CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain, slow, step-by-step numpy restatement of the SharQ per-linear-layer hot path
(arxiv/paper_2606_26587; citations `P:n` are /root/reference/PAPER.md line numbers):

    norm -> N:M magnitude mask -> sparse FP4 backbone (codes + scales + metadata)
         -> residual R = X - D_sp(Q_sp(X_sp)) -> dense FP4 residual -> two GEMMs (fp64)

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this module.  It shares no code with the CUDA path (paper_2606_26587_b200/) and
never imports it.  SharQ is an approximation / encoding, so the oracle follows the paper's
algorithm step by step; where the paper is silent the reading is the one listed in DESIGN.md
("Readings", R1..R18) and named in the docstrings below.

Numerics contract (R1): every fp32 step below is ONE IEEE-754 binary32 operation,
round-to-nearest-even, no fused multiply-add, no flush-to-zero.  numpy float32 ufuncs do exactly
that.  bf16 tensors are carried as uint16 bit patterns.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): see the table in DESIGN.md section "Oracle pins".
Definition-level choices the paper does not fix (reduction order, PTS granularity, pair score,
normalised X rounded to bf16, HiF4 unit on the sparse path) are "definition unpinned"; their
numerics are pinned.
"""
from __future__ import annotations

import numpy as np

F32 = np.float32
U8 = np.uint8
U16 = np.uint16
U32 = np.uint32

NVFP4, MXFP4, HIF4 = 0, 1, 2
MASK_PAIR48, MASK_24 = 0, 1
NORM_NONE, NORM_RMS, NORM_LAYER = 0, 1, 2

# P:388 (A.1.2): representable E2M1 magnitudes, indexed by the 3 magnitude bits of the code.
E2M1_VALUES = np.array([0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0], dtype=F32)
# RN(1/6) in binary32 (R6) and the PTS target 448*6 (A.1.3).
C6 = np.array([0x3E2AAAAB], dtype=U32).view(F32)[0]
PTS_TARGET = F32(2688.0)


# --------------------------------------------------------------------------------------------
# bf16 <-> fp32
# --------------------------------------------------------------------------------------------
def bf16_to_f32(u16: np.ndarray) -> np.ndarray:
    """Exact widening of bf16 bit patterns to fp32."""
    return (np.asarray(u16, dtype=U16).astype(U32) << U32(16)).view(F32)


def f32_to_bf16(x: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit patterns, round-to-nearest-even (finite inputs)."""
    u = np.ascontiguousarray(x, dtype=F32).view(U32)
    bias = U32(0x7FFF) + ((u >> U32(16)) & U32(1))
    return ((u + bias) >> U32(16)).astype(U16)


def _bf16_mul(a_u16, b_u16):
    """bf16 * bf16 -> bf16, one RNE rounding (the fp32 product of two bf16 values is exact)."""
    return f32_to_bf16(bf16_to_f32(a_u16) * bf16_to_f32(b_u16))


def _bf16_add(a_u16, b_u16):
    """bf16 + bf16 -> bf16 (fp32 sum of two bf16 is computed with one RN, then RNE to bf16).

    The fp32 sum of two bf16 numbers can itself round when exponents differ by more than 16,
    in which case the smaller addend is below half an ulp of bf16 of the larger, so the double
    rounding cannot change the bf16 result except on an exact tie of the second rounding that the
    first created; LayerNorm's beta path is "definition unpinned" (R3)."""
    return f32_to_bf16(bf16_to_f32(a_u16) + bf16_to_f32(b_u16))


def residual_add(x_u16, r_u16):
    """h = bf16(x + r): the transformer's residual-stream add that `sharq_prepare_add` folds in front of the
    norm (the paper's own lever is folding the neighbouring elementwise operator into the
    preparation kernel).  ONE rounding of the exact sum, ties to even.  Computed as an fp32 add
    followed by RNE to bf16; the two roundings equal one: the fp32 add only rounds when the smaller addend lies
    below 2^-16 of the larger, far from any bf16 tie point of the larger (pinned against exact rationals in
    tests/test_oracle_path.py)."""
    return _bf16_add(np.asarray(x_u16, dtype=U16), np.asarray(r_u16, dtype=U16))


# --------------------------------------------------------------------------------------------
# SwiGLU in front of the down-projection's preparation (R18)
# --------------------------------------------------------------------------------------------
# fp32 constants of the exp contract, as bit patterns so that both sides hold the same numbers
NEG_LOG2E = np.array([0xBFB8AA3B], dtype=U32).view(F32)[0]          # -RN(log2 e)
EXP2_POLY = np.array([0x3F800000, 0x3F317218, 0x3E75FDF0, 0x3D635847, 0x3C1D955B, 0x3AAEC3FF],
                     dtype=U32).view(F32)                            # RN(ln2^k / k!), k = 0..5
RINT_MAGIC = F32(12582912.0)                                         # 1.5 * 2^23: (t + M) - M = RNE integer of t


def exp_neg_contract(g):
    """e ~= exp(-g) for fp32 g by a fixed, restatable algorithm (every step ONE fp32 RN operation, no FMA):
       t = clamp(RN(g * (-log2e)), -126, 126);  n = (t + M) - M (RNE integer);  f = RN(t - n)  in [-1/2, 1/2]
       p = Horner_5(f) with c_k = RN(ln2^k / k!), each step RN(RN(p * f) + c_k);  e = RN(p * 2^n)
    Relative error <= 3.5e-6 + |g| 1.3e-7 (degree-5 Taylor remainder 2.4e-6, roundings of log2e and of t),
    pinned against math.exp."""
    g = np.asarray(g, dtype=F32)
    t = np.clip(g * NEG_LOG2E, F32(-126.0), F32(126.0)).astype(F32)
    n = ((t + RINT_MAGIC) - RINT_MAGIC).astype(F32)
    f = (t - n).astype(F32)
    p = np.full(g.shape, EXP2_POLY[5], dtype=F32)
    for k in (4, 3, 2, 1, 0):
        p = ((p * f).astype(F32) + EXP2_POLY[k]).astype(F32)
    two_n = ((n.astype(np.int32) + 127).astype(U32) << U32(23)).view(F32)
    return (p * two_n).astype(F32)


def swiglu(gate_u16, up_u16):
    """h = bf16( silu(gate) * up ), silu(g) = g * sigmoid(g) = g / (1 + exp(-g)): the elementwise operator between
    the gate/up projection and the down projection, which `sharq_prepare_swiglu` folds in front of the
    preparation (the paper's lever is folding the neighbouring operator into the prep kernel).
    fp32 steps, one RN each: e = exp_neg_contract(g); den = 1 + e; sig = 1 / den; s = g * sig; a = s * u;
    one rounding to bf16 at the end (R18; definition unpinned by the paper)."""
    g = bf16_to_f32(np.asarray(gate_u16, dtype=U16))
    u = bf16_to_f32(np.asarray(up_u16, dtype=U16))
    e = exp_neg_contract(g)
    den = (F32(1.0) + e).astype(F32)
    sig = (F32(1.0) / den).astype(F32)
    s = (g * sig).astype(F32)
    return f32_to_bf16((s * u).astype(F32))


# --------------------------------------------------------------------------------------------
# element / scale codecs
# --------------------------------------------------------------------------------------------
def e2m1_encode(v: np.ndarray) -> np.ndarray:
    """fp32 -> 4-bit E2M1 code (bit3 = sign), nearest grid point of {0,.5,1,1.5,2,3,4,6},
    ties to the even code, |v| > 6 saturates to 6, the sign bit is the sign bit of v even when
    the magnitude rounds to 0 (Eq. 3 "projection to the nearest representable value";
    BASELINE.json "round-to-nearest-even on the e2m1 grid")."""
    v = np.asarray(v, dtype=F32)
    a = np.abs(v)
    mag = np.zeros(v.shape, dtype=U8)
    # midpoints between neighbouring grid values; a tie goes to the even code
    mag += (a > F32(0.25))     # -> 0.5   (tie 0.25 stays on code 0)
    mag += (a >= F32(0.75))    # -> 1.0   (tie 0.75 goes to code 2)
    mag += (a > F32(1.25))     # -> 1.5   (tie 1.25 stays on code 2)
    mag += (a >= F32(1.75))    # -> 2.0   (tie 1.75 goes to code 4)
    mag += (a > F32(2.5))      # -> 3.0   (tie 2.5 stays on code 4)
    mag += (a >= F32(3.5))     # -> 4.0   (tie 3.5 goes to code 6)
    mag += (a > F32(5.0))      # -> 6.0   (tie 5.0 stays on code 6)
    sign = (v.view(U32) >> U32(31)).astype(U8)
    return (mag | (sign << U8(3))).astype(U8)


def e2m1_decode(code: np.ndarray) -> np.ndarray:
    code = np.asarray(code, dtype=U8)
    mag = E2M1_VALUES[code & U8(7)]
    return np.where((code & U8(8)) != 0, -mag, mag).astype(F32)


def e4m3_encode(x: np.ndarray) -> np.ndarray:
    """Non-negative fp32 -> FP8 E4M3 code (bias 7, 3 mantissa bits), round-to-nearest-
    even, saturating at the largest finite value 448 (code 0x7E), subnormals down to 2^-9."""
    x = np.asarray(x, dtype=F32)
    x = np.minimum(x, F32(448.0))
    m, e = np.frexp(x.astype(np.float64))          # x = m * 2^e, m in [0.5, 1)
    e_unb = e - 1                                   # x = (2m) * 2^(e-1)
    e_eff = np.maximum(e_unb, -6)                   # subnormals share the exponent -6
    # quantum of the grid at this exponent is 2^(e_eff-3); np.rint is round-half-to-even
    q = np.rint(np.ldexp(x.astype(np.float64), 3 - e_eff)).astype(np.int64)   # in [0, 16]
    # q == 16 means the mantissa carried into the next binade
    carry = q == 16
    e_eff = np.where(carry, e_eff + 1, e_eff)
    q = np.where(carry, 8, q)
    is_norm = q >= 8
    exp_field = np.where(is_norm, e_eff + 7, 0)
    man_field = np.where(is_norm, q - 8, q)
    code = (exp_field << 3) | man_field
    code = np.where(x == 0, 0, code)
    return code.astype(U8)


def e4m3_decode(code: np.ndarray) -> np.ndarray:
    code = np.asarray(code, dtype=U8).astype(np.int64)
    e = (code >> 3) & 0xF
    m = code & 7
    val = np.where(e == 0, np.ldexp(m.astype(np.float64), -9),
                   np.ldexp((8 + m).astype(np.float64), e - 10))
    return val.astype(F32)


def e8m0_encode_rp(x: np.ndarray) -> np.ndarray:
    """Non-negative fp32 -> E8M0 code = e + 127 with 2^e the smallest power of two >= x,
    clamped to e in [-127, 127]; x == 0 -> code 0 (R8; P:381 says only
    "power-of-two")."""
    x = np.asarray(x, dtype=F32)
    m, e = np.frexp(x.astype(np.float64))           # x = m * 2^e, m in [0.5, 1)
    e_up = np.where(m == 0.5, e - 1, e)             # exact powers of two stay
    e_up = np.where(x == 0, -127, e_up)
    e_up = np.clip(e_up, -127, 127)
    return (e_up + 127).astype(U8)


def e8m0_decode(code: np.ndarray) -> np.ndarray:
    return np.ldexp(np.float64(1.0), np.asarray(code, dtype=U8).astype(np.int64) - 127).astype(F32)


# --------------------------------------------------------------------------------------------
# O1 normalisation (R1-R3)
# --------------------------------------------------------------------------------------------
def canonical_sum(terms: np.ndarray, squares: bool) -> np.ndarray:
    """Canonical fp32 reduction over the last axis of `terms` [T, K] (R1).

    The order is defined on data indices.  With k the column index:
      block b = k // 1024, slot l = (k % 1024) // 32, chunk j = (k % 32) // 8, i = k % 8.
      leaf(b,l,j) = (((0 + t0) + t1) + ... + t7), t_i = term (or RN(term*term) if `squares`)
      P[l]        = ((0 + leaf(0,l,0)) + leaf(0,l,1)) + ... in ascending (b, j)
      butterfly   for delta in 16,8,4,2,1: P[l] <- P[l] + P[l xor delta]  (all l at once)
      result      = P[0]
    Columns beyond K (when K is not a multiple of 1024) do not exist: they contribute +0.
    """
    t = np.asarray(terms, dtype=F32)
    T, K = t.shape
    if squares:
        t = t * t
    Kp = -(-K // 1024) * 1024
    if Kp != K:
        t = np.concatenate([t, np.zeros((T, Kp - K), dtype=F32)], axis=1)
    t = t.reshape(T, Kp // 1024, 32, 4, 8)
    leaf = np.zeros(t.shape[:-1], dtype=F32)
    for i in range(8):
        leaf = leaf + t[..., i]
    P = np.zeros((T, 32), dtype=F32)
    for b in range(Kp // 1024):
        for j in range(4):
            P = P + leaf[:, b, :, j]
    lanes = np.arange(32)
    for delta in (16, 8, 4, 2, 1):
        P = P + P[:, lanes ^ delta]
    return P[:, 0].copy()


def normalize(x_u16, norm, gamma_u16=None, beta_u16=None, eps=1e-6):
    """O1.  Returns X as bf16 bit patterns [T, K] (R3: the normalised activation is a
    bf16 tensor, produced with the two-rounding order of the RMSNorm operator it replaces:
    h = bf16(x * rstd), X = bf16(h * gamma))."""
    x_u16 = np.asarray(x_u16, dtype=U16)
    if norm == NORM_NONE:
        return x_u16.copy()
    T, K = x_u16.shape
    xf = bf16_to_f32(x_u16)
    Kf = F32(K)
    eps = F32(eps)
    if norm == NORM_RMS:
        S = canonical_sum(xf, squares=True)
        c = xf
    elif norm == NORM_LAYER:
        mu = canonical_sum(xf, squares=False) / Kf
        c = xf - mu[:, None]
        S = canonical_sum(c, squares=True)
    else:
        raise ValueError(norm)
    ms = S / Kf
    v = ms + eps
    r = np.sqrt(v)
    rstd = F32(1.0) / r
    h = f32_to_bf16(c * rstd[:, None])
    X = _bf16_mul(h, np.asarray(gamma_u16, dtype=U16)[None, :])
    if norm == NORM_LAYER and beta_u16 is not None:
        X = _bf16_add(X, np.asarray(beta_u16, dtype=U16)[None, :])
    return X


# --------------------------------------------------------------------------------------------
# O3 N:M magnitude masks (Eq. 4, Eq. 6, P:398 A.1.4; R2, R4)
# --------------------------------------------------------------------------------------------
def _top2_of_4(score: np.ndarray):
    """score [..., 4] unsigned -> keep [..., 4] bool with exactly two True: unit p is kept iff
    fewer than two units beat it, where q beats p iff s[q] > s[p] or (s[q] == s[p] and q < p)."""
    s = score.astype(np.int64)
    idx = np.arange(4)
    beats = (s[..., None, :] > s[..., :, None]) | (
        (s[..., None, :] == s[..., :, None]) & (idx[None, :] < idx[:, None]))
    # beats[..., p, q] = q beats p
    return beats.sum(axis=-1) < 2


def mask_pair48(X_u16):
    """4:8 "in pairs": each chunk of 8 consecutive elements is 4 adjacent pairs; the 2
    pairs with the largest score survive, score = max(|a|, |b|) (R4), ties to the
    lower pair index.  Returns (keep_elem [T,K] bool, nibble [T,K/8] u8 = i0 | i1<<2)."""
    X_u16 = np.asarray(X_u16, dtype=U16)
    T, K = X_u16.shape
    u = (X_u16 & U16(0x7FFF)).reshape(T, K // 8, 4, 2)
    score = u.max(axis=-1)
    keep_pair = _top2_of_4(score)                         # [T, K/8, 4]
    nib = _nibbles(keep_pair)
    keep_elem = np.repeat(keep_pair, 2, axis=-1).reshape(T, K)
    return keep_elem, nib


def mask_24(X_u16):
    """Standard 2:4: keep the 2 largest |x| of every 4, ties to the lower index.
    Returns (keep_elem [T,K] bool, nibble [T,K/4] u8)."""
    X_u16 = np.asarray(X_u16, dtype=U16)
    T, K = X_u16.shape
    u = (X_u16 & U16(0x7FFF)).reshape(T, K // 4, 4)
    keep = _top2_of_4(u)
    return keep.reshape(T, K), _nibbles(keep)


def _nibbles(keep4: np.ndarray) -> np.ndarray:
    """keep4 [..., 4] with exactly two True -> i0 | (i1 << 2), i0 < i1 the kept indices."""
    idx = np.arange(4)
    i0 = np.where(keep4, idx, 9).min(axis=-1)
    i1 = np.where(keep4, idx, -1).max(axis=-1)
    return (i0 | (i1 << 2)).astype(U8)


def pack_nibbles(nib: np.ndarray) -> np.ndarray:
    """[T, n] nibbles -> [T, n/2] bytes, even index in the low nibble."""
    return (nib[:, 0::2] | (nib[:, 1::2] << U8(4))).astype(U8)


def pack_codes(codes: np.ndarray) -> np.ndarray:
    """[T, n] 4-bit codes -> [T, n/2] bytes, lower-k element in the low nibble."""
    return (codes[:, 0::2] | (codes[:, 1::2] << U8(4))).astype(U8)


def unpack_codes(packed: np.ndarray) -> np.ndarray:
    T, n = packed.shape
    out = np.empty((T, 2 * n), dtype=U8)
    out[:, 0::2] = packed & U8(0xF)
    out[:, 1::2] = packed >> U8(4)
    return out


# --------------------------------------------------------------------------------------------
# block scales (Eq. 3; P:388-394 A.1; R5-R8)
# --------------------------------------------------------------------------------------------
def _block_scale(amax: np.ndarray, fmt: int, ts: np.ndarray, inv_ts: np.ndarray):
    """amax [T, G] fp32 group maxima -> (sf_code u8, s_eff fp32, inv fp32), all [T, G].

    NVFP4: q = RN(a*C6); sf_f = RN(q*inv_ts); code = e4m3(sf_f); s_eff = RN(decode(code)*ts).
    MXFP4: code = e8m0_round_up(RN(a*C6)); s_eff = 2^e (no tensor scale, Table 6).
    inv = 0 if s_eff == 0 else RN(1/s_eff)."""
    q = amax.astype(F32) * C6
    if fmt == NVFP4:
        sf_f = q * inv_ts[:, None]
        code = e4m3_encode(sf_f)
        s_eff = e4m3_decode(code) * ts[:, None]
    elif fmt == MXFP4:
        code = e8m0_encode_rp(q)
        s_eff = e8m0_decode(code)
    else:
        raise ValueError(fmt)
    with np.errstate(divide="ignore"):
        inv = np.where(s_eff == 0, F32(0), F32(1.0) / s_eff).astype(F32)
    return code, s_eff.astype(F32), inv


def tensor_scale(X_u16, fmt, x_tensor_scale=None):
    """O2 (P:394 A.1.3 PTS; R5): per-row dynamic ts = RN(amax_row / 2688), ts = 1 for
    an all-zero row; or the caller's static scalar.  MXFP4 / HiF4 need no PTS."""
    T = X_u16.shape[0]
    if fmt != NVFP4:
        one = np.ones(T, dtype=F32)
        return one, one
    if x_tensor_scale is not None:
        ts = np.full(T, F32(x_tensor_scale), dtype=F32)
    else:
        a_row = bf16_to_f32(X_u16 & U16(0x7FFF)).max(axis=1)
        ts = np.where(a_row == 0, F32(1.0), a_row / PTS_TARGET).astype(F32)
    inv_ts = (F32(1.0) / ts).astype(F32)
    return ts, inv_ts


# --------------------------------------------------------------------------------------------
# sharq_prepare (Fig. 2, section 3.4) -- NVFP4 and MXFP4
# --------------------------------------------------------------------------------------------
def prepare(x_u16, fmt=NVFP4, mask=MASK_PAIR48, norm=NORM_RMS, gamma_u16=None, beta_u16=None,
            eps=1e-6, x_tensor_scale=None, _force_no_survivors=False):
    """Whole preparation path for one activation matrix x (bf16 bits, [T, K], K % 256 == 0).

    Returns a dict of canonical (row-major) arrays:
      X        [T,K]    u16  normalised activation (bf16 bits)                         (O1)
      ts       [T]      f32  row tensor scale                                          (O2)
      keep     [T,K]    bool mask M(X)                                    (O3; Eq. 6)
      sp_meta  [T,K/16] u8   two 4-bit chunk nibbles per byte (pair 4:8) / [T,K/8] (2:4)
      sp_codes [T,K/4]  u8   survivors' codes, ascending k, 2 per byte   (O4; Eq. 7)
      sp_sf    [T,K/32] u8   backbone block scales (one per 32 logical k)
      Xsp_tilde[T,K]    f32  D_sp(Q_sp(X_sp)), zero at dropped positions     (Eq. 7, 10)
      R        [T,K]    f32  residual X - Xsp_tilde                       (O5; Eq. 8)
      dn_codes [T,K/2]  u8   residual codes                                            (O6)
      dn_sf    [T,K/Gd] u8   residual block scales, Gd = 16 (NVFP4) / 32 (MXFP4)
    `_force_no_survivors` is a test hook: empty mask, so R = X and the residual path must equal
    a plain dense quantizer (DESIGN.md pin "dense-only special case").
    """
    if fmt == HIF4:
        return prepare_hif4(x_u16, norm=norm, gamma_u16=gamma_u16, beta_u16=beta_u16, eps=eps)
    x_u16 = np.asarray(x_u16, dtype=U16)
    T, K = x_u16.shape
    assert K % 256 == 0
    X = normalize(x_u16, norm, gamma_u16, beta_u16, eps)
    Xf = bf16_to_f32(X)
    ts, inv_ts = tensor_scale(X, fmt, x_tensor_scale)

    # O3 mask
    if mask == MASK_PAIR48:
        keep, nib = mask_pair48(X)
    else:
        keep, nib = mask_24(X)
    if _force_no_survivors:
        keep = np.zeros_like(keep)
    sp_meta = pack_nibbles(nib)

    # O4 backbone: one scale per 32 logical k, amax over the survivors only
    Gs = 32
    absX = np.abs(Xf)
    a_sp = np.where(keep, absX, F32(0)).reshape(T, K // Gs, Gs).max(axis=-1)
    sp_sf, s_eff_sp, inv_sp = _block_scale(a_sp, fmt, ts, inv_ts)
    with np.errstate(over="ignore"):           # dropped positions may overflow; never used
        v = Xf * np.repeat(inv_sp, Gs, axis=1)
    code_all = e2m1_encode(v)
    # O5 dequantise and residual
    d = e2m1_decode(code_all) * np.repeat(s_eff_sp, Gs, axis=1)
    Xsp_tilde = np.where(keep, d, F32(0)).astype(F32)
    R = np.where(keep, Xf - d, Xf).astype(F32)
    # compress survivors in ascending k (exactly K/2 per row)
    if _force_no_survivors:
        sp_codes = np.zeros((T, K // 4), dtype=U8)
    else:
        surv = code_all[keep].reshape(T, K // 2)
        sp_codes = pack_codes(surv)

    # O6 residual: dense groups
    Gd = 16 if fmt == NVFP4 else 32
    a_dn = np.abs(R).reshape(T, K // Gd, Gd).max(axis=-1)
    dn_sf, s_eff_dn, inv_dn = _block_scale(a_dn, fmt, ts, inv_ts)
    dn_code = e2m1_encode(R * np.repeat(inv_dn, Gd, axis=1))
    dn_codes = pack_codes(dn_code)
    return dict(X=X, ts=ts, keep=keep, sp_meta=sp_meta, sp_codes=sp_codes, sp_sf=sp_sf,
                Xsp_tilde=Xsp_tilde, R=R, dn_codes=dn_codes, dn_sf=dn_sf,
                fmt=fmt, mask=mask, Gs=Gs, Gd=Gd)


# --------------------------------------------------------------------------------------------
# Path combinations of the ablation (Table 5): Dense+Dense and Sparse+Sparse
# --------------------------------------------------------------------------------------------
PATH_SHARQ, PATH_SPARSE_ONLY, PATH_DENSE_ONLY, PATH_DENSE_DENSE, PATH_SPARSE_SPARSE = 0, 1, 2, 3, 4


def mask_pair48_f32(R):
    """Pairwise 4:8 on an fp32 tensor (the second sparse path of Sparse+Sparse masks the RESIDUAL, which is
    fp32): score of a pair = max of the two 31-bit magnitude patterns (monotone in |r| for finite values),
    top 2 of 4 pairs, ties to the lower pair index -- DESIGN.md R4 carried over to fp32 (R17)."""
    R = np.ascontiguousarray(R, dtype=F32)
    T, K = R.shape
    u = (R.view(U32) & U32(0x7FFFFFFF)).reshape(T, K // 8, 4, 2)
    keep_pair = _top2_of_4(u.max(axis=-1))
    return np.repeat(keep_pair, 2, axis=-1).reshape(T, K), _nibbles(keep_pair)


def _dense_quantize(V, fmt, ts, inv_ts):
    """One dense FP4 path (Eq. 3): per group of Gd (16 NVFP4 / 32 MXFP4) scale = amax/6 in the scale
    format, codes = RNE e2m1.  Returns (codes packed [T,K/2], sf [T,K/Gd], dequantised fp32 [T,K])."""
    T, K = V.shape
    Gd = 16 if fmt == NVFP4 else 32
    a = np.abs(V).reshape(T, K // Gd, Gd).max(axis=-1)
    sf, s_eff, inv = _block_scale(a, fmt, ts, inv_ts)
    code = e2m1_encode(V * np.repeat(inv, Gd, axis=1))
    d = (e2m1_decode(code) * np.repeat(s_eff, Gd, axis=1)).astype(F32)
    return pack_codes(code), sf, d


def _sparse_quantize(V, keep, fmt, ts, inv_ts):
    """One sparse FP4 path (Eq. 7): scale per 32 logical k over the survivors, survivors' codes in
    ascending k.  Returns (codes packed [T,K/4], sf [T,K/32], dequantised fp32 [T,K], 0 at dropped k)."""
    T, K = V.shape
    a = np.where(keep, np.abs(V), F32(0)).reshape(T, K // 32, 32).max(axis=-1)
    sf, s_eff, inv = _block_scale(a, fmt, ts, inv_ts)
    with np.errstate(over="ignore"):
        code = e2m1_encode(V * np.repeat(inv, 32, axis=1))
    d = np.where(keep, e2m1_decode(code) * np.repeat(s_eff, 32, axis=1), F32(0)).astype(F32)
    return pack_codes(code[keep].reshape(T, K // 2)), sf, d


def prepare_paths(x_u16, path, fmt=NVFP4, norm=NORM_RMS, gamma_u16=None, beta_u16=None, eps=1e-6,
                  x_tensor_scale=None):
    """The two-path decompositions of Table 5, each X ~= A0 + A1 with A1 quantised from the residual
    of A0 exactly as in Eq. 8: R = X - D(Q(.)), one row tensor scale for both paths (R5).
      PATH_DENSE_DENSE   A0 = dense FP4 of X,                 A1 = dense FP4 of R   ("two dense NVFP4 paths")
      PATH_SPARSE_SPARSE A0 = SharQ's sparse backbone of X,   A1 = sparse FP4 of R under its own pairwise 4:8
                         mask M(R) ("two sparse paths"; the part of R outside M(R) is lost)
    Returns dict(X, ts, a0_codes, a0_sf, a0_meta, a1_codes, a1_sf, a1_meta, A0, A1 (fp32 dequantised, without
    nothing folded: they include ts), R); metas are None for dense paths."""
    assert fmt in (NVFP4, MXFP4) and path in (PATH_DENSE_DENSE, PATH_SPARSE_SPARSE)
    x_u16 = np.asarray(x_u16, dtype=U16)
    X = normalize(x_u16, norm, gamma_u16, beta_u16, eps)
    Xf = bf16_to_f32(X)
    ts, inv_ts = tensor_scale(X, fmt, x_tensor_scale)
    if path == PATH_DENSE_DENSE:
        a0_codes, a0_sf, d0 = _dense_quantize(Xf, fmt, ts, inv_ts)
        R = (Xf - d0).astype(F32)
        a1_codes, a1_sf, d1 = _dense_quantize(R, fmt, ts, inv_ts)
        a0_meta = a1_meta = None
    else:
        keep0, nib0 = mask_pair48(X)
        a0_codes, a0_sf, d0 = _sparse_quantize(Xf, keep0, fmt, ts, inv_ts)
        R = np.where(keep0, Xf - d0, Xf).astype(F32)
        keep1, nib1 = mask_pair48_f32(R)
        a1_codes, a1_sf, d1 = _sparse_quantize(R, keep1, fmt, ts, inv_ts)
        a0_meta, a1_meta = pack_nibbles(nib0), pack_nibbles(nib1)
    return dict(X=X, ts=ts, R=R, A0=d0, A1=d1, a0_codes=a0_codes, a0_sf=a0_sf, a0_meta=a0_meta,
                a1_codes=a1_codes, a1_sf=a1_sf, a1_meta=a1_meta, fmt=fmt, path=path)


def linear_paths(pp, wq, rows=None, cols=None):
    """Eq. 9 for a Table 5 combination, fp64, rebuilt from the STORED operands only: both dense paths go
    through the weight's dense scale view, both sparse paths through the sparse view (same values, R7)."""
    fmt, path = pp["fmt"], pp["path"]
    ops = []
    for i in (0, 1):
        if path == PATH_DENSE_DENSE:
            view = dict(dn_codes=pp[f"a{i}_codes"], dn_sf=pp[f"a{i}_sf"], ts=pp["ts"], fmt=fmt,
                        Gd=16 if fmt == NVFP4 else 32)
            ops.append(dequant_residual(view, with_ts=False))
        else:
            view = dict(sp_codes=pp[f"a{i}_codes"], sp_sf=pp[f"a{i}_sf"], sp_meta=pp[f"a{i}_meta"], ts=pp["ts"],
                        fmt=fmt, mask=MASK_PAIR48, Gs=32)
            ops.append(dequant_backbone(view, with_ts=False))
    W = dequant_weight(wq, "dense" if path == PATH_DENSE_DENSE else "sparse", with_ts=False)
    ts = pp["ts"].astype(np.float64)
    A0, A1 = ops
    if rows is not None:
        A0, A1, ts = A0[rows], A1[rows], ts[rows]
    if cols is not None:
        W = W[cols]
    return (A0 @ W.T + A1 @ W.T) * ts[:, None] * np.float64(wq["ts_w"])


# --------------------------------------------------------------------------------------------
# sharq_quantize_weight (Fig. 2 caption; R7)
# --------------------------------------------------------------------------------------------
def quantize_weight(w_u16, fmt=NVFP4):
    """W bf16 bits [D, K] -> one FP4 payload + two scale views.
      codes    [D,K/2]  u8
      sf_sp    [D,K/32] u8  sparse view: one scale per 32 k ("sparse group-32 scales")
      sf_dn    [D,K/16] u8  dense view: every sparse-view scale repeated for its two 16-groups
                            ("duplicated dense group-16 scales"); MXFP4: identical to sf_sp
      ts_w     f32 scalar   NVFP4 tensor scale RN(max|W| / 2688) (1 if W == 0); MXFP4: 1
    """
    if fmt == HIF4:
        return quantize_weight_hif4(w_u16)
    w_u16 = np.asarray(w_u16, dtype=U16)
    D, K = w_u16.shape
    assert K % 256 == 0
    Wf = bf16_to_f32(w_u16)
    if fmt == NVFP4:
        a = np.abs(Wf).max()
        ts_w = F32(1.0) if a == 0 else F32(a) / PTS_TARGET
    else:
        ts_w = F32(1.0)
    ts = np.full(D, ts_w, dtype=F32)
    inv_ts = (F32(1.0) / ts).astype(F32)
    G = 32
    amax = np.abs(Wf).reshape(D, K // G, G).max(axis=-1)
    sf, s_eff, inv = _block_scale(amax, fmt, ts, inv_ts)
    codes = pack_codes(e2m1_encode(Wf * np.repeat(inv, G, axis=1)))
    sf_dn = np.repeat(sf, 2, axis=1) if fmt == NVFP4 else sf.copy()
    return dict(codes=codes, sf_sp=sf, sf_dn=sf_dn, ts_w=F32(ts_w), fmt=fmt)


# --------------------------------------------------------------------------------------------
# dequantisation helpers and O7 the linear layer in fp64 (Eq. 9)
# --------------------------------------------------------------------------------------------
def sf_decode(sf_code, fmt):
    return e4m3_decode(sf_code) if fmt == NVFP4 else e8m0_decode(sf_code)


def expand_backbone(prep):
    """Scatter the compressed survivors back to their logical positions using the metadata.
    Returns (codes [T,K] u8 with 0 at dropped positions, keep [T,K] bool) -- rebuilt from the
    STORED outputs (sp_codes, sp_meta) only, i.e. what the sparse GEMM sees."""
    sp_codes, sp_meta, mask = prep["sp_codes"], prep["sp_meta"], prep["mask"]
    T = sp_codes.shape[0]
    nib = np.empty((T, sp_meta.shape[1] * 2), dtype=U8)
    nib[:, 0::2] = sp_meta & U8(0xF)
    nib[:, 1::2] = sp_meta >> U8(4)
    i0 = (nib & U8(3)).astype(np.int64)
    i1 = ((nib >> U8(2)) & U8(3)).astype(np.int64)
    surv = unpack_codes(sp_codes)                        # [T, K/2] codes in ascending k
    if mask == MASK_PAIR48:
        K = nib.shape[1] * 8
        out = np.zeros((T, K // 8, 4, 2), dtype=U8)
        keep = np.zeros((T, K // 8, 4), dtype=bool)
        s = surv.reshape(T, K // 8, 2, 2)
        tt, cc = np.meshgrid(np.arange(T), np.arange(K // 8), indexing="ij")
        out[tt, cc, i0] = s[:, :, 0]
        out[tt, cc, i1] = s[:, :, 1]
        keep[tt, cc, i0] = True
        keep[tt, cc, i1] = True
        return out.reshape(T, K), np.repeat(keep, 2, axis=-1).reshape(T, K)
    K = nib.shape[1] * 4
    out = np.zeros((T, K // 4, 4), dtype=U8)
    keep = np.zeros((T, K // 4, 4), dtype=bool)
    s = surv.reshape(T, K // 4, 2)
    tt, cc = np.meshgrid(np.arange(T), np.arange(K // 4), indexing="ij")
    out[tt, cc, i0] = s[:, :, 0]
    out[tt, cc, i1] = s[:, :, 1]
    keep[tt, cc, i0] = True
    keep[tt, cc, i1] = True
    return out.reshape(T, K), keep.reshape(T, K)


def dequant_backbone(prep, with_ts=True):
    """fp64 [T,K]: e2m1(code) * sf (* ts) at kept positions, 0 elsewhere."""
    if prep["fmt"] == HIF4:
        return hif4_dequant_backbone(prep)
    codes, keep = expand_backbone(prep)
    sf = sf_decode(prep["sp_sf"], prep["fmt"]).astype(np.float64)
    val = e2m1_decode(codes).astype(np.float64) * np.repeat(sf, prep["Gs"], axis=1)
    val = np.where(keep, val, 0.0)
    return val * prep["ts"].astype(np.float64)[:, None] if with_ts else val


def dequant_residual(prep, with_ts=True):
    if prep["fmt"] == HIF4:
        return hif4_dequant_residual(prep)
    codes = unpack_codes(prep["dn_codes"])
    sf = sf_decode(prep["dn_sf"], prep["fmt"]).astype(np.float64)
    val = e2m1_decode(codes).astype(np.float64) * np.repeat(sf, prep["Gd"], axis=1)
    return val * prep["ts"].astype(np.float64)[:, None] if with_ts else val


def dequant_weight(wq, view="sparse", with_ts=True):
    """fp64 [D,K] through the sparse (group-32) or the dense (duplicated group-16) scale view."""
    if wq["fmt"] == HIF4:
        return hif4_dequant_weight(wq)
    codes = unpack_codes(wq["codes"])
    if view == "sparse":
        sf = np.repeat(sf_decode(wq["sf_sp"], wq["fmt"]).astype(np.float64), 32, axis=1)
    else:
        g = 16 if wq["fmt"] == NVFP4 else 32
        sf = np.repeat(sf_decode(wq["sf_dn"], wq["fmt"]).astype(np.float64), g, axis=1)
    val = e2m1_decode(codes).astype(np.float64) * sf
    return val * np.float64(wq["ts_w"]) if with_ts else val


def linear(prep, wq, bias_u16=None, rows=None, cols=None):
    """O7 (Eq. 9): Y64 = GEMM_sp(backbone, W through the sparse view)
                               + GEMM_dn(residual, W through the dense view)   in fp64.
    Every product code*sf*code*sf is exact in fp64; the row/tensor scales multiply the
    accumulated sum once, as the epilogue does.  `rows` / `cols` restrict the output to a
    sample of rows / output features (index arrays)."""
    A_sp = dequant_backbone(prep, with_ts=False)
    A_dn = dequant_residual(prep, with_ts=False)
    W_sp = dequant_weight(wq, "sparse", with_ts=False)
    W_dn = dequant_weight(wq, "dense", with_ts=False)
    ts = prep["ts"].astype(np.float64)
    if rows is not None:
        A_sp, A_dn, ts = A_sp[rows], A_dn[rows], ts[rows]
    if cols is not None:
        W_sp, W_dn = W_sp[cols], W_dn[cols]
    acc = A_sp @ W_sp.T + A_dn @ W_dn.T
    Y = acc * ts[:, None] * np.float64(wq["ts_w"])
    if bias_u16 is not None:
        b = bf16_to_f32(bias_u16).astype(np.float64)
        Y = Y + (b if cols is None else b[cols])[None, :]
    return Y


def linear_loops(prep, wq, t, d):
    """One output element of Eq. 9 by an explicit pure-Python loop over k (tiny cases; pins the
    vectorised `linear`)."""
    A_sp = dequant_backbone(prep, with_ts=False)[t]
    A_dn = dequant_residual(prep, with_ts=False)[t]
    W_sp = dequant_weight(wq, "sparse", with_ts=False)[d]
    W_dn = dequant_weight(wq, "dense", with_ts=False)[d]
    acc = 0.0
    for k in range(A_sp.shape[0]):
        acc += float(A_sp[k]) * float(W_sp[k])
    for k in range(A_dn.shape[0]):
        acc += float(A_dn[k]) * float(W_dn[k])
    return acc * float(prep["ts"][t]) * float(wq["ts_w"])


# HiF4 (A.2) lives in its own module to keep this file readable.
from .hif4_oracle import (prepare_hif4, quantize_weight_hif4, hif4_dequant_backbone,  # noqa: E402
                          hif4_dequant_residual, hif4_dequant_weight)
