// sharq_prepare: the fused activation-preparation kernel (Fig. 2).
//
// One warp owns one activation row at a time.  The row is brought into shared memory with 16-byte
// cp.async copies (coalesced 512-byte warp requests, XOR-swizzled destination), then every lane
// works on 32 CONTIGUOUS elements of each 1024-element block: one backbone scale group (32), two
// residual scale groups (16) and four 4:8 mask chunks (8) all live inside one lane, so the mask,
// both amax reductions, the sparse compression and the residual need no shuffles at all; the only
// cross-lane steps are the per-row butterflies (sum of squares, row amax).  Outputs leave as
// 16/8/2/1-byte stores that are contiguous across the warp.
//
// Numerics follow DESIGN.md R1-R8 exactly (the oracle in oracle/ restates them in numpy); every
// rounding is an explicit *_rn intrinsic so no FMA contraction can change a bit.
#include <cuda_fp16.h>
#include <stdlib.h>

#include "common.cuh"
#include "debug_env.h"

namespace sharq {

struct PrepParams {
  const uint16_t* x; int64_t ldx; int64_t T; int64_t K;
  const uint16_t* gamma; const uint16_t* beta; const float* x_ts;
  uint8_t* sp_codes; uint8_t* sp_sf; uint8_t* sp_meta; uint8_t* dn_codes; uint8_t* dn_sf; float* row_scale;
  float eps; int tiled; int nbuf; uint32_t row_bytes;
};

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// 16-byte chunk q of a row lives at chunk position q ^ ((q >> 3) & 3): lane l reading its four
// chunks 4l+s hits 8 distinct 16-byte bank groups per quarter-warp.
__device__ __forceinline__ uint32_t swz(uint32_t q) { return q ^ ((q >> 3) & 3u); }

__device__ __forceinline__ void issue_row_load(const PrepParams& p, int64_t row, uint32_t buf, int lane) {
  const uint8_t* src = reinterpret_cast<const uint8_t*>(p.x + row * p.ldx);
  const uint32_t nchunk = (uint32_t)(p.K >> 3);
  for (uint32_t q = lane; q < nchunk; q += 32) cp_async16(buf + swz(q) * 16, src + (size_t)q * 16);
}

__device__ __forceinline__ void lds_block(uint32_t buf, uint32_t blk, int lane, uint32_t (&v)[16]) {
  const uint32_t r = (lane >> 1) & 3u;
  const uint32_t base = buf + (blk * 128u + lane * 4u) * 16u;
#pragma unroll
  for (int s = 0; s < 4; ++s) {
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v[4 * s]), "=r"(v[4 * s + 1]), "=r"(v[4 * s + 2]), "=r"(v[4 * s + 3])
                 : "r"(base + ((s ^ r) << 4)));
  }
}
__device__ __forceinline__ void sts_block(uint32_t buf, uint32_t blk, int lane, const uint32_t (&v)[16]) {
  const uint32_t r = (lane >> 1) & 3u;
  const uint32_t base = buf + (blk * 128u + lane * 4u) * 16u;
#pragma unroll
  for (int s = 0; s < 4; ++s) {
    asm volatile("st.shared.v4.u32 [%4], {%0,%1,%2,%3};" ::"r"(v[4 * s]), "r"(v[4 * s + 1]), "r"(v[4 * s + 2]),
                 "r"(v[4 * s + 3]), "r"(base + ((s ^ r) << 4))
                 : "memory");
  }
}

__device__ __forceinline__ float warp_sum_butterfly(float v) {
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) v = __fadd_rn(v, __shfl_xor_sync(0xffffffffu, v, d));
  return v;
}
__device__ __forceinline__ uint32_t warp_max_u32(uint32_t v) {
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, d));
  return v;
}

// canonical leaf (R1): (((0 + t0) + t1) + ... + t7) over one 8-chunk, t = x*x or x.
template <bool SQ>
__device__ __forceinline__ float leaf8(const uint32_t* v) {
  float acc = 0.0f;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    float lo = bf16lo_to_f32(v[i]), hi = bf16hi_to_f32(v[i]);
    if (SQ) {  // lo*lo is exact in fp32 (bf16 operand), so fma == mul then add
      acc = __fmaf_rn(lo, lo, acc);
      acc = __fmaf_rn(hi, hi, acc);
    } else {
      acc = __fadd_rn(acc, lo);
      acc = __fadd_rn(acc, hi);
    }
  }
  return acc;
}

// x * y >> 32 as an integer multiply (FMA pipe): the ALU pipe is the kernel's bottleneck
__device__ __forceinline__ uint32_t mulhi_u32(uint32_t x, uint32_t y) {
  uint32_t r;
  asm("mul.hi.u32 %0, %1, %2;" : "=r"(r) : "r"(x), "r"(y));
  return r;
}

// top-2-of-4 on keys (score << 2 | 3 - p): returns nibble i0 | i1 << 2 and the best key.
__device__ __forceinline__ void top2of4(uint32_t k0, uint32_t k1, uint32_t k2, uint32_t k3, uint32_t& i0,
                                        uint32_t& i1, uint32_t& best) {
  uint32_t m01 = max(k0, k1), n01 = min(k0, k1), m23 = max(k2, k3), n23 = min(k2, k3);
  uint32_t t1 = max(m01, m23);
  // second largest of two sorted pairs: the smaller group maximum or the larger group minimum
  uint32_t t2 = max(min(m01, m23), max(n01, n23));
  uint32_t a = (t1 & 3u) ^ 3u, b = (t2 & 3u) ^ 3u;
  i0 = min(a, b);
  i1 = max(a, b);
  best = t1;
}

struct BlockScale { uint32_t code; float s_eff; float inv; };

template <int FMT>
__device__ __forceinline__ BlockScale block_scale(float amax, float ts, float inv_ts) {
  BlockScale r;
  const float q = __fmul_rn(amax, __uint_as_float(0x3E2AAAABu));  // RN(a * RN(1/6))
  if (FMT == SHARQ_NVFP4) {
    const float sf_f = __fmul_rn(q, inv_ts);
    r.code = cvt_e4m3(sf_f);
    r.s_eff = __fmul_rn(e4m3_to_f32(r.code), ts);
    r.inv = (r.s_eff == 0.0f) ? 0.0f : __frcp_rn(r.s_eff);
  } else {
    r.code = e8m0_round_up(q);
    r.s_eff = e8m0_to_f32(r.code);
    r.inv = e8m0_inv_to_f32(r.code);
  }
  return r;
}

__device__ __forceinline__ uint32_t mullo_u32(uint32_t x, uint32_t y) {   // x * y on the FMA pipe (no shift)
  uint32_t r;
  asm("mul.lo.u32 %0, %1, %2;" : "=r"(r) : "r"(x), "r"(y));
  return r;
}

// O3 for one lane's 32 elements: what the later steps need from the mask, small enough to stay in registers
// across the row-scale reduction.  sel[w] is the byte-permute selector that compresses chunks 2w and 2w+1
// (nibbles: i0, i1 of chunk 2w, then 4 + i0, 4 + i1 of chunk 2w+1); keep bit 4c+q = pair q of chunk c
// survives; amax_bits = the largest bf16 magnitude of the lane's block (the best pair of a chunk is always
// kept, so this is both the backbone group amax and the lane's share of the row amax).
struct MaskSel { uint32_t sel[2]; uint32_t keep; uint32_t meta16; uint32_t amax_bits; };

__device__ __forceinline__ void mask_block_e2m1(const uint32_t (&X)[16], MaskSel& ms) {
  ms.sel[0] = ms.sel[1] = 0u;
  ms.keep = 0u; ms.meta16 = 0u; ms.amax_bits = 0u;
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    uint32_t key[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      // the sign bits fall off the top: the upper 15 bits of x << 17 / x << 1 are |lo| / |hi|; their
      // unsigned maximum has max(|lo|, |hi|) in its upper 15 bits.  Shifts as multiplies: FMA pipe.
      const uint32_t m = max(mullo_u32(X[4 * c + q], 131072u), mullo_u32(X[4 * c + q], 2u));
      key[q] = mullo_u32(mulhi_u32(m, 32768u), 4u) + (3u - q);
    }
    uint32_t i0, i1, best;
    top2of4(key[0], key[1], key[2], key[3], i0, i1, best);
    ms.amax_bits = max(ms.amax_bits, best >> 2);
    ms.keep |= ((1u << i0) | (1u << i1)) << (4 * c);
    ms.meta16 |= (i0 | (i1 << 2)) << (4 * c);
    const uint32_t two = (c & 1) ? (i0 | (i1 << 4)) + 0x44u : (i0 | (i1 << 4));
    ms.sel[c >> 1] |= two << (8 * (c & 1));
  }
}

// One lane, 32 contiguous elements X[16] (packed bf16 pairs): backbone, residual, stores (O4-O7).
template <int FMT>
__device__ __forceinline__ void quantize_tail_e2m1(const PrepParams& p, int64_t row, uint32_t k0,
                                                   const uint32_t (&X)[16], const MaskSel& ms, float ts,
                                                   float inv_ts) {
  // ---- O4 backbone scale over the 16 survivors of this 32-group
  const BlockScale bs = block_scale<FMT>(__uint_as_float(ms.amax_bits << 16), ts, inv_ts);

  float R[32];
  uint32_t bytes[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    float xs[8];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      xs[2 * q] = bf16lo_to_f32(X[4 * c + q]);
      xs[2 * q + 1] = bf16hi_to_f32(X[4 * c + q]);
    }
    // all four pairs of the chunk in one word: byte q = the two codes of pair q
    bytes[c] = cvt_e2m1x8(__fmul_rn(xs[0], bs.inv), __fmul_rn(xs[1], bs.inv), __fmul_rn(xs[2], bs.inv),
                          __fmul_rn(xs[3], bs.inv), __fmul_rn(xs[4], bs.inv), __fmul_rn(xs[5], bs.inv),
                          __fmul_rn(xs[6], bs.inv), __fmul_rn(xs[7], bs.inv));
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      // ---- O5 dequantise and residual; a dropped pair keeps R = X bit for bit
      float dl, dh;
      e2m1x2_to_f32((bytes[c] >> (8 * q)) & 0xFFu, dl, dh);
      float rl = xs[2 * q], rh = xs[2 * q + 1];
      if (ms.keep & (1u << (4 * c + q))) {
        rl = __fsub_rn(rl, __fmul_rn(dl, bs.s_eff));
        rh = __fsub_rn(rh, __fmul_rn(dh, bs.s_eff));
      }
      R[8 * c + 2 * q] = rl;
      R[8 * c + 2 * q + 1] = rh;
    }
  }
  // compress: survivors in ascending k; one byte permute per two chunks
  uint32_t sp_word[2];
  sp_word[0] = __byte_perm(bytes[0], bytes[1], ms.sel[0]);
  sp_word[1] = __byte_perm(bytes[2], bytes[3], ms.sel[1]);
  const uint32_t meta16 = ms.meta16;

  // ---- O6 residual: NVFP4 two groups of 16, MXFP4 one group of 32
  uint32_t dn_word[4];
  uint32_t dn_sf[2];
  constexpr int GD = (FMT == SHARQ_NVFP4) ? 16 : 32;
#pragma unroll
  for (int g = 0; g < 32 / GD; ++g) {
    float a = 0.0f;
#pragma unroll
    for (int i = 0; i < GD; ++i) a = fmaxf(a, fabsf(R[g * GD + i]));
    const BlockScale ds = block_scale<FMT>(a, ts, inv_ts);
    dn_sf[g] = ds.code;
#pragma unroll
    for (int w = 0; w < GD / 8; ++w) {
      const int e = g * GD + w * 8;
      dn_word[g * (GD / 8) + w] =
          cvt_e2m1x8(__fmul_rn(R[e], ds.inv), __fmul_rn(R[e + 1], ds.inv), __fmul_rn(R[e + 2], ds.inv),
                     __fmul_rn(R[e + 3], ds.inv), __fmul_rn(R[e + 4], ds.inv), __fmul_rn(R[e + 5], ds.inv),
                     __fmul_rn(R[e + 6], ds.inv), __fmul_rn(R[e + 7], ds.inv));
    }
  }

  // ---- O7 stores (k0 = first logical k of this lane's block)
  const int64_t K = p.K;
  *reinterpret_cast<uint2*>(p.sp_codes + row * (K >> 2) + (k0 >> 2)) = make_uint2(sp_word[0], sp_word[1]);
  *reinterpret_cast<uint4*>(p.dn_codes + row * (K >> 1) + (k0 >> 1)) =
      make_uint4(dn_word[0], dn_word[1], dn_word[2], dn_word[3]);
  const int64_t g32 = k0 >> 5;
  if (p.tiled) {
    *reinterpret_cast<uint16_t*>(p.sp_meta + meta_tiled_offset(row, 2 * g32, K)) = (uint16_t)meta16;
    p.sp_sf[sf_tiled_offset(row, g32, K >> 5)] = (uint8_t)bs.code;
    if (FMT == SHARQ_NVFP4)
      *reinterpret_cast<uint16_t*>(p.dn_sf + sf_tiled_offset(row, 2 * g32, K >> 4)) =
          (uint16_t)(dn_sf[0] | (dn_sf[1] << 8));
    else
      p.dn_sf[sf_tiled_offset(row, g32, K >> 5)] = (uint8_t)dn_sf[0];
  } else {
    *reinterpret_cast<uint16_t*>(p.sp_meta + row * (K >> 4) + 2 * g32) = (uint16_t)meta16;
    p.sp_sf[row * (K >> 5) + g32] = (uint8_t)bs.code;
    if (FMT == SHARQ_NVFP4)
      *reinterpret_cast<uint16_t*>(p.dn_sf + row * (K >> 4) + 2 * g32) = (uint16_t)(dn_sf[0] | (dn_sf[1] << 8));
    else
      p.dn_sf[row * (K >> 5) + g32] = (uint8_t)dn_sf[0];
  }
}

template <int FMT>
__device__ __forceinline__ void quantize_block_e2m1(const PrepParams& p, int64_t row, uint32_t k0,
                                                    const uint32_t (&X)[16], float ts, float inv_ts) {
  MaskSel ms;
  mask_block_e2m1(X, ms);
  quantize_tail_e2m1<FMT>(p, row, k0, X, ms, ts, inv_ts);
}

// ---- HiF4: Algorithm 1 on a 64-element unit shared by two lanes (32 elements each) -------
struct Hif4Scale { uint32_t e6m2; float base; float rec; };

// SF (a non-negative bf16 value held in fp32) -> E6M2 code, its value and the table reciprocal
__device__ __forceinline__ Hif4Scale hif4_scale(float vmax) {
  // line 10: SF = bf16(Vmax * (1/7)_bf16)
  const uint32_t sfb = mul_bf16x2_rn(__float_as_uint(vmax) >> 16, 0x3E12u) & 0xFFFFu;
  const float sf = __uint_as_float(sfb << 16);
  int E = (int)(sfb >> 7) - 127;
  uint32_t m7 = sfb & 0x7Fu, m2 = m7 >> 5, rem = m7 & 31u;
  m2 += (rem > 16u || (rem == 16u && (m2 & 1u))) ? 1u : 0u;   // RNE to 2 mantissa bits (R9)
  if (m2 == 4u) { m2 = 0u; E += 1; }
  int code = ((E + 48) << 2) | (int)m2;
  if (sf < __uint_as_float(0x27800000u)) code = 0;             // < 2^-48 (includes 0)
  if (sf > 49152.0f || E + 48 > 63) code = 0xFE;               // > 2^15 * 1.5
  Hif4Scale r;
  r.e6m2 = (uint32_t)code;
  const int Ec = (code >> 2) - 48;
  const uint32_t mc = (uint32_t)code & 3u;
  r.base = __uint_as_float(((uint32_t)(Ec + 127) << 23) | (mc << 21));
  const uint32_t lut = (mc == 0u) ? 0x3F800000u : (mc == 1u) ? 0x3F4D0000u : (mc == 2u) ? 0x3F2B0000u : 0x3F120000u;
  r.rec = __uint_as_float(lut - ((uint32_t)Ec << 23));
  return r;
}

// Quantise 32 bf16 values V (packed pairs) of a unit whose scale is `hs`; v16[8] are the per-4 maxima.
// Returns 32 S1P2 codes in c[4] (8 nibbles per word), E1_8 bits (4) and E1_16 bits (8), and the decoded
// values d[32] (Eq. 15) when WANT_D.
template <bool WANT_D>
__device__ __forceinline__ void hif4_quant32(const uint32_t (&V)[16], const float (&v16)[8], const Hif4Scale& hs,
                                             uint32_t (&c)[4], uint32_t& e8bits, uint32_t& e16bits, float* d) {
  e8bits = 0; e16bits = 0;
#pragma unroll
  for (int g = 0; g < 4; ++g) {                                  // one E1_8 group = 8 elements
    const float v8 = fmaxf(v16[2 * g], v16[2 * g + 1]);
    const bool e8 = __fmul_rn(v8, hs.rec) >= 4.0f;               // line 13
    const float s8 = e8 ? 0.5f : 1.0f;
    e8bits |= (e8 ? 1u : 0u) << g;
    uint32_t word = 0;
#pragma unroll
    for (int h = 0; h < 2; ++h) {                                // one E1_16 group = 4 elements
      const bool e16 = __fmul_rn(__fmul_rn(v16[2 * g + h], hs.rec), s8) >= 2.0f;   // line 14
      const float s16 = e16 ? 0.5f : 1.0f;
      e16bits |= (e16 ? 1u : 0u) << (2 * g + h);
      const float up = hs.base * (e8 ? 2.0f : 1.0f) * (e16 ? 2.0f : 1.0f);         // exact power-of-two products
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const uint32_t pk = V[4 * g + 2 * h + j];
        const uint32_t sb = pack_bf16x2_rn(__fmul_rn(bf16lo_to_f32(pk), hs.rec), __fmul_rn(bf16hi_to_f32(pk), hs.rec));
        const float sl = __fmul_rn(__fmul_rn(bf16lo_to_f32(sb), s8), s16);          // line 19
        const float sh = __fmul_rn(__fmul_rn(bf16hi_to_f32(sb), s8), s16);
        const uint32_t ml = (uint32_t)min(__float2int_rn(__fmul_rn(fabsf(sl), 4.0f)), 7);
        const uint32_t mh = (uint32_t)min(__float2int_rn(__fmul_rn(fabsf(sh), 4.0f)), 7);
        const uint32_t cl = ml | ((__float_as_uint(sl) >> 28) & 8u), ch = mh | ((__float_as_uint(sh) >> 28) & 8u);
        word |= (cl | (ch << 4)) << (8 * (2 * h + j));
        if (WANT_D) {
          const float vl = __fmul_rn((float)ml * 0.25f, up), vh = __fmul_rn((float)mh * 0.25f, up);
          d[8 * g + 4 * h + 2 * j] = (cl & 8u) ? -vl : vl;
          d[8 * g + 4 * h + 2 * j + 1] = (ch & 8u) ? -vh : vh;
        }
      }
    }
    c[g] = word;
  }
}

__device__ __forceinline__ uint32_t hif4_meta_word(uint32_t e6m2, uint32_t e8bits, uint32_t e16bits, int lane) {
  const uint32_t part = (e8bits << (8 + 4 * (lane & 1))) | (e16bits << (16 + 8 * (lane & 1)));
  return e6m2 | part | __shfl_xor_sync(0xffffffffu, part, 1);
}

__device__ __forceinline__ void quantize_block_hif4(const PrepParams& p, int64_t row, uint32_t k0,
                                                    const uint32_t (&X)[16], int lane, bool active) {
  // ---- 2:4 mask per 4 elements, M (.) X with +0 at dropped positions
  uint32_t Xs[16], nibs = 0;
  float v16[8];
  uint32_t keepbits = 0;
#pragma unroll
  for (int g = 0; g < 8; ++g) {
    const uint32_t a0 = X[2 * g] & 0x7FFF7FFFu, a1 = X[2 * g + 1] & 0x7FFF7FFFu;
    uint32_t i0, i1, best;
    top2of4(((a0 & 0xFFFFu) << 2) | 3u, ((a0 >> 16) << 2) | 2u, ((a1 & 0xFFFFu) << 2) | 1u, ((a1 >> 16) << 2) | 0u,
            i0, i1, best);
    nibs |= (i0 | (i1 << 2)) << (4 * g);
    const uint32_t kb = (1u << i0) | (1u << i1);
    keepbits |= kb << (4 * g);
    Xs[2 * g] = X[2 * g] & (((kb & 1u) ? 0xFFFFu : 0u) | ((kb & 2u) ? 0xFFFF0000u : 0u));
    Xs[2 * g + 1] = X[2 * g + 1] & (((kb & 4u) ? 0xFFFFu : 0u) | ((kb & 8u) ? 0xFFFF0000u : 0u));
    v16[g] = __uint_as_float((best >> 2) << 16);
  }
  float vmax = 0.0f;
#pragma unroll
  for (int g = 0; g < 8; ++g) vmax = fmaxf(vmax, v16[g]);
  vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, 1));
  const Hif4Scale hs = hif4_scale(vmax);
  uint32_t c[4], e8b, e16b;
  float d[32];
  hif4_quant32<true>(Xs, v16, hs, c, e8b, e16b, d);
  const uint32_t sp_meta_word = hif4_meta_word(hs.e6m2, e8b, e16b, lane);
  // compress survivors: per 4 elements keep nibbles i0, i1 (ascending)
  uint32_t spw[2] = {0u, 0u};
#pragma unroll
  for (int g = 0; g < 8; ++g) {
    const uint32_t four = (c[g >> 1] >> (16 * (g & 1))) & 0xFFFFu;
    const uint32_t i0 = (nibs >> (4 * g)) & 3u, i1 = (nibs >> (4 * g + 2)) & 3u;
    const uint32_t byte = ((four >> (4 * i0)) & 0xFu) | (((four >> (4 * i1)) & 0xFu) << 4);
    spw[g >> 2] |= byte << (8 * (g & 3));
  }
  // ---- residual R = X - d (kept) / X (dropped), rounded to bf16 for Alg. 1
  uint32_t Rb[16];
  float r16[8];
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const float dl = ((keepbits >> (2 * i)) & 1u) ? d[2 * i] : 0.0f;
    const float dh = ((keepbits >> (2 * i + 1)) & 1u) ? d[2 * i + 1] : 0.0f;
    Rb[i] = pack_bf16x2_rn(__fsub_rn(bf16lo_to_f32(X[i]), dl), __fsub_rn(bf16hi_to_f32(X[i]), dh));
  }
  float rmax = 0.0f;
#pragma unroll
  for (int g = 0; g < 8; ++g) {
    const uint32_t a0 = Rb[2 * g] & 0x7FFF7FFFu, a1 = Rb[2 * g + 1] & 0x7FFF7FFFu;
    const uint32_t m = max(max(a0 & 0xFFFFu, a0 >> 16), max(a1 & 0xFFFFu, a1 >> 16));
    r16[g] = __uint_as_float(m << 16);
    rmax = fmaxf(rmax, r16[g]);
  }
  rmax = fmaxf(rmax, __shfl_xor_sync(0xffffffffu, rmax, 1));
  const Hif4Scale hd = hif4_scale(rmax);
  uint32_t cd[4], f8b, f16b;
  hif4_quant32<false>(Rb, r16, hd, cd, f8b, f16b, nullptr);
  const uint32_t dn_meta_word = hif4_meta_word(hd.e6m2, f8b, f16b, lane);
  if (!active) return;
  const int64_t K = p.K;
  *reinterpret_cast<uint2*>(p.sp_codes + row * (K >> 2) + (k0 >> 2)) = make_uint2(spw[0], spw[1]);
  *reinterpret_cast<uint4*>(p.dn_codes + row * (K >> 1) + (k0 >> 1)) = make_uint4(cd[0], cd[1], cd[2], cd[3]);
  *reinterpret_cast<uint32_t*>(p.sp_meta + row * (K >> 3) + (k0 >> 3)) = nibs;
  if ((lane & 1) == 0) {
    reinterpret_cast<uint32_t*>(p.sp_sf)[row * (K >> 6) + (k0 >> 6)] = sp_meta_word;
    reinterpret_cast<uint32_t*>(p.dn_sf)[row * (K >> 6) + (k0 >> 6)] = dn_meta_word;
  }
}

// ---- the kernel ------------------------------------------------------------------------------------
template <int FMT, int NORM>
__global__ void __launch_bounds__(512) sharq_prepare_kernel(const PrepParams p) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  const int64_t gwarp = (int64_t)blockIdx.x * nwarps + warp, gstride = (int64_t)gridDim.x * nwarps;
  const uint32_t wbase = smem_u32(smem_raw) + (uint32_t)warp * p.nbuf * p.row_bytes;
  const int64_t K = p.K;
  const uint32_t nblk = (uint32_t)((K + 1023) >> 10);
  const float Kf = (float)K;
  const float static_ts = (FMT == SHARQ_NVFP4 && p.x_ts != nullptr) ? *p.x_ts : 0.0f;

  int64_t row = gwarp;
  if (row < p.T) issue_row_load(p, row, wbase, lane);
  cp_async_commit();
  uint32_t cur = 0;
  for (; row < p.T; row += gstride) {
    const uint32_t buf = wbase + cur * p.row_bytes;
    if (p.nbuf == 2) {  // prefetch the next row into the other buffer
      if (row + gstride < p.T) issue_row_load(p, row + gstride, wbase + (cur ^ 1u) * p.row_bytes, lane);
      cp_async_commit();
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncwarp();

    // ---- O1 normalisation statistics (canonical order, R1)
    float rstd = 1.0f, mu = 0.0f;
    if (NORM != SHARQ_NORM_NONE) {
      if (NORM == SHARQ_NORM_LAYER) {
        float acc = 0.0f;
        for (uint32_t b = 0; b < nblk; ++b) {
          uint32_t v[16];
          const bool act = (int64_t)b * 1024 + lane * 32 < K;
          if (act) lds_block(buf, b, lane, v);
#pragma unroll
          for (int c = 0; c < 4; ++c) acc = __fadd_rn(acc, act ? leaf8<false>(&v[4 * c]) : 0.0f);
        }
        mu = __fdiv_rn(warp_sum_butterfly(acc), Kf);
      }
      float acc = 0.0f;
      for (uint32_t b = 0; b < nblk; ++b) {
        uint32_t v[16];
        const bool act = (int64_t)b * 1024 + lane * 32 < K;
        if (act) lds_block(buf, b, lane, v);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          float leaf = 0.0f;
          if (act) {
            if (NORM == SHARQ_NORM_RMS) {
              leaf = leaf8<true>(&v[4 * c]);
            } else {
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                const float cl = __fsub_rn(bf16lo_to_f32(v[4 * c + i]), mu), ch = __fsub_rn(bf16hi_to_f32(v[4 * c + i]), mu);
                leaf = __fadd_rn(leaf, __fmul_rn(cl, cl));
                leaf = __fadd_rn(leaf, __fmul_rn(ch, ch));
              }
            }
          }
          acc = __fadd_rn(acc, leaf);
        }
      }
      const float S = warp_sum_butterfly(acc);
      rstd = __frcp_rn(__fsqrt_rn(__fadd_rn(__fdiv_rn(S, Kf), p.eps)));
    }

    // ---- normalise in place (h = bf16(c * rstd), X = bf16(h * gamma) [+ beta]) and the row amax (O2)
    float ts = 1.0f, inv_ts = 1.0f;
    const bool need_rowmax = (FMT == SHARQ_NVFP4) && (p.x_ts == nullptr);
    if (NORM != SHARQ_NORM_NONE || need_rowmax) {
      uint32_t amax = 0;
      for (uint32_t b = 0; b < nblk; ++b) {
        const int64_t k0 = (int64_t)b * 1024 + lane * 32;
        if (k0 >= K) continue;
        uint32_t v[16];
        lds_block(buf, b, lane, v);
        if (NORM != SHARQ_NORM_NONE) {
          const uint4* g4 = reinterpret_cast<const uint4*>(p.gamma + k0);
          const uint4* b4 = (NORM == SHARQ_NORM_LAYER && p.beta) ? reinterpret_cast<const uint4*>(p.beta + k0) : nullptr;
#pragma unroll
          for (int s = 0; s < 4; ++s) {
            const uint4 g = __ldg(g4 + s);
            const uint32_t gg[4] = {g.x, g.y, g.z, g.w};
            uint32_t bb[4] = {0u, 0u, 0u, 0u};
            if (b4) { const uint4 t = __ldg(b4 + s); bb[0] = t.x; bb[1] = t.y; bb[2] = t.z; bb[3] = t.w; }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              float lo = bf16lo_to_f32(v[4 * s + i]), hi = bf16hi_to_f32(v[4 * s + i]);
              if (NORM == SHARQ_NORM_LAYER) { lo = __fsub_rn(lo, mu); hi = __fsub_rn(hi, mu); }
              const uint32_t h = pack_bf16x2_rn(__fmul_rn(lo, rstd), __fmul_rn(hi, rstd));
              uint32_t X = mul_bf16x2_rn(h, gg[i]);
              if (b4) X = add_bf16x2_rn(X, bb[i]);
              v[4 * s + i] = X;
            }
          }
          sts_block(buf, b, lane, v);
        }
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          const uint32_t a = v[i] & 0x7FFF7FFFu;
          amax = max(amax, max(a & 0xFFFFu, a >> 16));
        }
      }
      if (need_rowmax) {
        amax = warp_max_u32(amax);
        const float a_row = __uint_as_float(amax << 16);
        ts = (amax == 0u) ? 1.0f : __fdiv_rn(a_row, 2688.0f);
      }
    }
    if (FMT == SHARQ_NVFP4) {
      if (p.x_ts != nullptr) ts = static_ts;
      inv_ts = __frcp_rn(ts);
    }
    if (lane == 0) p.row_scale[row] = ts;

    // ---- mask, backbone, residual, stores: 32 contiguous elements per lane per 1024-block
    for (uint32_t b = 0; b < nblk; ++b) {
      const int64_t k0 = (int64_t)b * 1024 + lane * 32;
      const bool act = k0 < K;
      uint32_t X[16];
      if (act) {
        lds_block(buf, b, lane, X);
      } else {
#pragma unroll
        for (int i = 0; i < 16; ++i) X[i] = 0u;
      }
      if (FMT == SHARQ_HIF4) {
        quantize_block_hif4(p, row, (uint32_t)k0, X, lane, act);
      } else if (act) {
        quantize_block_e2m1<FMT>(p, row, (uint32_t)k0, X, ts, inv_ts);
      }
    }
    __syncwarp();   // all lanes are done with `buf` before it is refilled
    if (p.nbuf == 2) {
      cur ^= 1u;
    } else {
      if (row + gstride < p.T) issue_row_load(p, row + gstride, buf, lane);
      cp_async_commit();
    }
  }
  cp_async_wait<0>();
}

// ---- row-per-CTA kernel (NVFP4 / MXFP4, K <= 32768) ---------------------------------------------------
// Warp w of the CTA owns the 1024-element block w of the row and every lane keeps its 32 contiguous
// elements in registers from the first load to the last store: no shared-memory staging of the row, so
// occupancy is set by registers only and a single row (decode, T = 1) is spread over K/1024 warps.  The
// row statistics keep DESIGN.md R1's order: every lane publishes its four 8-chunk leaves, warp 0 adds
// them in ascending (block, chunk) order per lane slot and runs the butterfly; the result is broadcast.
constexpr int kRowMaxWarps = 32;

// dynamic shared memory: leaf[nwarps][4][32] floats, then amax[32] words, then one float
struct RowShared {
  float* leaf;
  uint32_t* amax;
  float* stat;
};

// `slot` alternates between consecutive reductions so that the values of one reduction are never
// overwritten before every warp has read them: two barriers per reduction, none after the read.
__device__ __forceinline__ float row_reduce_ordered(RowShared& sh, const float (&leaf)[4], int warp, int lane,
                                                    int nwarps, uint32_t& slot) {
  float* buf = sh.leaf + (size_t)slot * nwarps * 128;
#pragma unroll
  for (int j = 0; j < 4; ++j) buf[(warp * 4 + j) * 32 + lane] = leaf[j];
  __syncthreads();
  if (warp == 0) {
    float acc = 0.0f;
    for (int b = 0; b < nwarps; ++b) {
#pragma unroll
      for (int j = 0; j < 4; ++j) acc = __fadd_rn(acc, buf[(b * 4 + j) * 32 + lane]);
    }
    acc = warp_sum_butterfly(acc);
    if (lane == 0) sh.stat[slot] = acc;
  }
  __syncthreads();
  const float r = sh.stat[slot];
  slot ^= 1u;
  return r;
}

template <int FMT, int NORM, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) sharq_prepare_row_kernel(const PrepParams p) {
  extern __shared__ __align__(16) uint8_t row_smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  RowShared sh;
  sh.leaf = reinterpret_cast<float*>(row_smem);                                   // [2][nwarps][4][32]
  sh.amax = reinterpret_cast<uint32_t*>(row_smem + (size_t)nwarps * 1024);        // [2][32]
  sh.stat = reinterpret_cast<float*>(row_smem + (size_t)nwarps * 1024 + 256);     // [2]
  uint32_t red_slot = 0, amax_slot = 0;
  // programmatic dependent launch: let the GEMM that follows start streaming its weights now; our own
  // inputs (and the operand buffers we overwrite) belong to the kernels before us
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  const int64_t K = p.K;
  const uint32_t k0 = (uint32_t)warp * 1024u + (uint32_t)lane * 32u;
  const bool act = (int64_t)k0 < K;
  const float Kf = (float)K;
  const float static_ts = (FMT == SHARQ_NVFP4 && p.x_ts != nullptr) ? *p.x_ts : 0.0f;
  const bool need_rowmax = (FMT == SHARQ_NVFP4) && (p.x_ts == nullptr);

  // gamma / beta of this lane's 32 columns: parked in shared memory as [4][threads] 16-byte words (conflict
  // free), not in registers: at 64 registers / thread the 16-32 words would spill to local memory
  uint4* g_sm = reinterpret_cast<uint4*>(row_smem + (size_t)nwarps * 1024 + 256 + 16);
  uint4* b_sm = g_sm + 4 * blockDim.x;
  if (NORM != SHARQ_NORM_NONE && act) {
    const uint4* g4 = reinterpret_cast<const uint4*>(p.gamma + k0);
#pragma unroll
    for (int s = 0; s < 4; ++s) g_sm[s * blockDim.x + threadIdx.x] = __ldg(g4 + s);
    if (NORM == SHARQ_NORM_LAYER && p.beta) {
      const uint4* b4 = reinterpret_cast<const uint4*>(p.beta + k0);
#pragma unroll
      for (int s = 0; s < 4; ++s) b_sm[s * blockDim.x + threadIdx.x] = __ldg(b4 + s);
    }
  }

  for (int64_t row = blockIdx.x; row < p.T; row += gridDim.x) {
    uint32_t X[16];
    if (act && (lane & 1) == 0 && row + gridDim.x < p.T)      // next row of this CTA: 128-byte line -> L2
      asm volatile("prefetch.global.L2 [%0];" ::"l"(p.x + (row + gridDim.x) * p.ldx + k0));
    if (act) {
      const uint4* src = reinterpret_cast<const uint4*>(p.x + row * p.ldx + k0);
#pragma unroll
      for (int s = 0; s < 4; ++s) {
        const uint4 v = __ldcs(src + s);
        X[4 * s] = v.x; X[4 * s + 1] = v.y; X[4 * s + 2] = v.z; X[4 * s + 3] = v.w;
      }
    } else {
#pragma unroll
      for (int i = 0; i < 16; ++i) X[i] = 0u;
    }

    // ---- O1 statistics in the canonical order (R1) and normalisation (R3)
    if (NORM != SHARQ_NORM_NONE) {
      float mu = 0.0f, leaf[4];
      if (NORM == SHARQ_NORM_LAYER) {
#pragma unroll
        for (int c = 0; c < 4; ++c) leaf[c] = act ? leaf8<false>(&X[4 * c]) : 0.0f;
        mu = __fdiv_rn(row_reduce_ordered(sh, leaf, warp, lane, nwarps, red_slot), Kf);
      }
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        float l = 0.0f;
        if (act) {
          if (NORM == SHARQ_NORM_RMS) {
            l = leaf8<true>(&X[4 * c]);
          } else {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const float cl = __fsub_rn(bf16lo_to_f32(X[4 * c + i]), mu), ch = __fsub_rn(bf16hi_to_f32(X[4 * c + i]), mu);
              l = __fadd_rn(l, __fmul_rn(cl, cl));
              l = __fadd_rn(l, __fmul_rn(ch, ch));
            }
          }
        }
        leaf[c] = l;
      }
      const float S = row_reduce_ordered(sh, leaf, warp, lane, nwarps, red_slot);
      const float rstd = __frcp_rn(__fsqrt_rn(__fadd_rn(__fdiv_rn(S, Kf), p.eps)));
      if (act) {
#pragma unroll
        for (int s4 = 0; s4 < 4; ++s4) {
          const uint4 gq = g_sm[s4 * blockDim.x + threadIdx.x];
          const uint32_t G[4] = {gq.x, gq.y, gq.z, gq.w};
          uint32_t Bt[4] = {0u, 0u, 0u, 0u};
          if (NORM == SHARQ_NORM_LAYER && p.beta) {
            const uint4 bq = b_sm[s4 * blockDim.x + threadIdx.x];
            Bt[0] = bq.x; Bt[1] = bq.y; Bt[2] = bq.z; Bt[3] = bq.w;
          }
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const int i = 4 * s4 + j;
            float lo = bf16lo_to_f32(X[i]), hi = bf16hi_to_f32(X[i]);
            if (NORM == SHARQ_NORM_LAYER) { lo = __fsub_rn(lo, mu); hi = __fsub_rn(hi, mu); }
            const uint32_t h = pack_bf16x2_rn(__fmul_rn(lo, rstd), __fmul_rn(hi, rstd));
            uint32_t v = mul_bf16x2_rn(h, G[j]);
            if (NORM == SHARQ_NORM_LAYER && p.beta) v = add_bf16x2_rn(v, Bt[j]);
            X[i] = v;
          }
        }
      }
    }

    // ---- O2 per-row tensor scale
    float ts = 1.0f, inv_ts = 1.0f;
    // the mask needs no scale: it runs first and its best pair scores give the lane's share of the row amax
    MaskSel ms;
    ms.amax_bits = 0u;
    if constexpr (FMT != SHARQ_HIF4) {
      if (act) mask_block_e2m1(X, ms);
    }
    if (need_rowmax) {
      uint32_t amax = warp_max_u32(ms.amax_bits);
      if (lane == 0) sh.amax[amax_slot * 32 + warp] = amax;
      __syncthreads();
      amax = warp_max_u32(lane < nwarps ? sh.amax[amax_slot * 32 + lane] : 0u);
      amax_slot ^= 1u;                           // the next row writes the other half: no second barrier
      ts = (amax == 0u) ? 1.0f : __fdiv_rn(__uint_as_float(amax << 16), 2688.0f);
    }
    if (FMT == SHARQ_NVFP4) {
      if (p.x_ts != nullptr) ts = static_ts;
      inv_ts = __frcp_rn(ts);
    }
    if (threadIdx.x == 0) p.row_scale[row] = ts;

    // ---- O3-O7 mask, backbone, residual, stores
    if constexpr (FMT == SHARQ_HIF4) {
      quantize_block_hif4(p, row, k0, X, lane, act);     // two lanes share a 64-element unit: all lanes take part
    } else {
      if (act) quantize_tail_e2m1<FMT>(p, row, k0, X, ms, ts, inv_ts);
    }
  }
}

template <int FMT>
static cudaError_t launch_row_kernel(int norm, const PrepParams& p, int num_sms, cudaStream_t st) {
  const int warps = (int)((p.K + 1023) / 1024);
  const dim3 block((unsigned)warps * 32);
  int per_sm = 2048 / (warps * 32);                       // thread limit; registers trim it further at launch
  if (debug_env().row_per_sm > 0) per_sm = debug_env().row_per_sm;
  if (per_sm < 1) per_sm = 1;
  if (per_sm > 32) per_sm = 32;                           // grid = about twice the resident CTAs (finer tail); 32 one-warp CTAs for short rows
  int64_t ctas = (int64_t)num_sms * per_sm;
  if (ctas > p.T) ctas = p.T;
  const dim3 grid((unsigned)ctas);
  cudaLaunchConfig_t lc{};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = debug_env().no_pdl ? 0 : 1;
  lc.gridDim = grid; lc.blockDim = block; lc.stream = st; lc.attrs = attr; lc.numAttrs = 1;
  lc.dynamicSmemBytes = (size_t)warps * 1024 + 256 + 16 + (norm != SHARQ_NORM_NONE ? (size_t)warps * 32 * 128 : 0);   // + gamma, beta
  cudaError_t err = cudaSuccess;
#define SHARQ_ROW(N, MAXT, MINB)                                                                              \
  do {                                                                                                        \
    auto kfn = sharq_prepare_row_kernel<FMT, N, MAXT, MINB>;                                                  \
    if (lc.dynamicSmemBytes > 48 * 1024)                                                                      \
      err = cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)lc.dynamicSmemBytes); \
    if (err == cudaSuccess) err = cudaLaunchKernelEx(&lc, kfn, p);                                            \
  } while (0)
#define SHARQ_ROW_N(MAXT, MINB)                                              \
  {                                                                          \
    if (norm == SHARQ_NORM_NONE) SHARQ_ROW(SHARQ_NORM_NONE, MAXT, MINB);     \
    else if (norm == SHARQ_NORM_RMS) SHARQ_ROW(SHARQ_NORM_RMS, MAXT, MINB);  \
    else SHARQ_ROW(SHARQ_NORM_LAYER, MAXT, MINB);                            \
  }
#ifndef SHARQ_ROW_MINB_128
#define SHARQ_ROW_MINB_128 8
#endif
#ifndef SHARQ_ROW_MINB_256
#define SHARQ_ROW_MINB_256 3
#endif
#ifndef SHARQ_ROW_MINB_512
#define SHARQ_ROW_MINB_512 2
#endif
  // occupancy beats register comfort here (measured: 64 registers with a few spills and 28-32 warps / SM is
  // up to 19 % faster than 96-128 registers with 14-20 warps: the kernel is issue bound with long stalls)
  if (warps <= 4) SHARQ_ROW_N(128, SHARQ_ROW_MINB_128)
  else if (warps <= 8) SHARQ_ROW_N(256, SHARQ_ROW_MINB_256)
  else if (warps <= 16) SHARQ_ROW_N(512, SHARQ_ROW_MINB_512)
  else SHARQ_ROW_N(1024, 1)                      // <= 64 registers
#undef SHARQ_ROW_N
#undef SHARQ_ROW
  return err;
}

template <int FMT>
static cudaError_t launch_norm(int norm, const PrepParams& p, dim3 grid, dim3 block, size_t smem, cudaStream_t st) {
#define SHARQ_LAUNCH(N)                                                                                        \
  {                                                                                                            \
    auto kfn = sharq_prepare_kernel<FMT, N>;                                                                   \
    cudaError_t e = cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);          \
    if (e != cudaSuccess) return e;                                                                            \
    kfn<<<grid, block, smem, st>>>(p);                                                                         \
    return cudaGetLastError();                                                                                 \
  }
  if (norm == SHARQ_NORM_NONE) SHARQ_LAUNCH(SHARQ_NORM_NONE)
  if (norm == SHARQ_NORM_RMS) SHARQ_LAUNCH(SHARQ_NORM_RMS)
  SHARQ_LAUNCH(SHARQ_NORM_LAYER)
#undef SHARQ_LAUNCH
}

// Host launcher, called by the C ABI in api.cu after argument validation.
cudaError_t launch_prepare(const sharq_config* cfg, const void* x, int64_t T, int64_t K, int64_t ldx,
                           const void* gamma, const void* beta, const float* x_ts, void* sp_codes, void* sp_sf,
                           void* sp_meta, void* dn_codes, void* dn_sf, float* row_scale, int num_sms,
                           cudaStream_t st) {
  PrepParams p;
  p.x = (const uint16_t*)x; p.ldx = ldx; p.T = T; p.K = K;
  p.gamma = (const uint16_t*)gamma; p.beta = (const uint16_t*)beta; p.x_ts = x_ts;
  p.sp_codes = (uint8_t*)sp_codes; p.sp_sf = (uint8_t*)sp_sf; p.sp_meta = (uint8_t*)sp_meta;
  p.dn_codes = (uint8_t*)dn_codes; p.dn_sf = (uint8_t*)dn_sf; p.row_scale = row_scale;
  p.eps = cfg->eps; p.tiled = (cfg->layout == SHARQ_LAYOUT_TILED);
  p.row_bytes = (uint32_t)(K * 2);
  if (K <= 1024 * kRowMaxWarps && !debug_env().old_prepare) {
    p.nbuf = 0;
    if (cfg->fmt == SHARQ_NVFP4) return launch_row_kernel<SHARQ_NVFP4>(cfg->norm, p, num_sms, st);
    if (cfg->fmt == SHARQ_MXFP4) return launch_row_kernel<SHARQ_MXFP4>(cfg->norm, p, num_sms, st);
    return launch_row_kernel<SHARQ_HIF4>(cfg->norm, p, num_sms, st);
  }
  // warps per CTA: as many double-buffered rows as fit in ~200 KB, else single-buffered
  const size_t budget = 200 * 1024;
  int nbuf = 2;
  int warps = (int)(budget / (2 * (size_t)p.row_bytes));
  if (warps < 8) { nbuf = 1; warps = (int)(budget / p.row_bytes); }
  if (warps > 16) warps = 16;
  if (warps < 1) return cudaErrorInvalidValue;
  p.nbuf = nbuf;
  int64_t ctas = (T + warps - 1) / warps;
  if (ctas > num_sms) ctas = num_sms;
  // few rows: spread them over more CTAs with fewer warps each
  if (T < (int64_t)num_sms * warps) { warps = (int)((T + num_sms - 1) / num_sms); ctas = (T + warps - 1) / warps; }
  const size_t smem = (size_t)warps * nbuf * p.row_bytes;
  dim3 grid((unsigned)ctas), block((unsigned)warps * 32);
  switch (cfg->fmt) {
    case SHARQ_NVFP4: return launch_norm<SHARQ_NVFP4>(cfg->norm, p, grid, block, smem, st);
    case SHARQ_MXFP4: return launch_norm<SHARQ_MXFP4>(cfg->norm, p, grid, block, smem, st);
    default: return launch_norm<SHARQ_HIF4>(cfg->norm, p, grid, block, smem, st);
  }
}

// ---- sharq_quantize_weight (offline): one payload, two scale views ---------------------
__global__ void weight_amax_kernel(const uint16_t* W, int64_t D, int64_t K, int64_t ldw, uint32_t* amax_bits) {
  uint32_t m = 0;
  const int64_t nvec = D * (K >> 3);
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t d = i / (K >> 3), c = i % (K >> 3);
    const uint4 v = __ldg(reinterpret_cast<const uint4*>(W + d * ldw + c * 8));
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) { const uint32_t a = w[j] & 0x7FFF7FFFu; m = max(m, max(a & 0xFFFFu, a >> 16)); }
  }
  m = warp_max_u32(m);
  if ((threadIdx.x & 31) == 0) atomicMax(amax_bits, m);
}

template <int FMT>
__global__ void weight_quant_kernel(const uint16_t* W, int64_t D, int64_t K, int64_t ldw, uint8_t* codes,
                                    uint8_t* sf_sp, uint8_t* sf_dn, float* ts_out, const uint32_t* amax_bits,
                                    int tiled) {
  const int lane = threadIdx.x & 31;
  const int64_t nblk = (K + 1023) >> 10;
  const int64_t item = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (item >= D * nblk) return;
  const int64_t d = item / nblk, b = item % nblk;
  float ts = 1.0f, inv_ts = 1.0f;
  if (FMT == SHARQ_NVFP4) {
    const uint32_t a = *amax_bits;
    ts = (a == 0u) ? 1.0f : __fdiv_rn(__uint_as_float(a << 16), 2688.0f);
    inv_ts = __frcp_rn(ts);
  }
  if (item == 0 && lane == 0) *ts_out = ts;
  const int64_t k0 = b * 1024 + lane * 32;
  const bool act = k0 < K;
  uint32_t X[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) X[i] = 0u;
  if (act) {
    const uint4* src = reinterpret_cast<const uint4*>(W + d * ldw + k0);
#pragma unroll
    for (int s = 0; s < 4; ++s) { const uint4 v = __ldg(src + s); X[4 * s] = v.x; X[4 * s + 1] = v.y; X[4 * s + 2] = v.z; X[4 * s + 3] = v.w; }
  }
  if (FMT == SHARQ_HIF4) {
    float v16[8], vmax = 0.0f;
#pragma unroll
    for (int g = 0; g < 8; ++g) {
      const uint32_t a0 = X[2 * g] & 0x7FFF7FFFu, a1 = X[2 * g + 1] & 0x7FFF7FFFu;
      v16[g] = __uint_as_float(max(max(a0 & 0xFFFFu, a0 >> 16), max(a1 & 0xFFFFu, a1 >> 16)) << 16);
      vmax = fmaxf(vmax, v16[g]);
    }
    vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, 1));
    const Hif4Scale hs = hif4_scale(vmax);
    uint32_t c[4], e8b, e16b;
    hif4_quant32<false>(X, v16, hs, c, e8b, e16b, nullptr);
    const uint32_t word = hif4_meta_word(hs.e6m2, e8b, e16b, lane);
    if (!act) return;
    *reinterpret_cast<uint4*>(codes + d * (K >> 1) + (k0 >> 1)) = make_uint4(c[0], c[1], c[2], c[3]);
    if ((lane & 1) == 0) {
      reinterpret_cast<uint32_t*>(sf_sp)[d * (K >> 6) + (k0 >> 6)] = word;
      reinterpret_cast<uint32_t*>(sf_dn)[d * (K >> 6) + (k0 >> 6)] = word;
    }
    return;
  }
  if (!act) return;
  uint32_t amax = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) { const uint32_t a = X[i] & 0x7FFF7FFFu; amax = max(amax, max(a & 0xFFFFu, a >> 16)); }
  const BlockScale bs = block_scale<FMT>(__uint_as_float(amax << 16), ts, inv_ts);
  uint32_t w[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    uint32_t word = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const uint32_t pk = X[4 * q + j];
      word |= cvt_e2m1x2(__fmul_rn(bf16lo_to_f32(pk), bs.inv), __fmul_rn(bf16hi_to_f32(pk), bs.inv)) << (8 * j);
    }
    w[q] = word;
  }
  *reinterpret_cast<uint4*>(codes + d * (K >> 1) + (k0 >> 1)) = make_uint4(w[0], w[1], w[2], w[3]);
  const int64_t g32 = k0 >> 5;
  const uint16_t dup = (uint16_t)(bs.code | (bs.code << 8));
  if (tiled) {
    sf_sp[sf_tiled_offset(d, g32, K >> 5)] = (uint8_t)bs.code;
    if (FMT == SHARQ_NVFP4) *reinterpret_cast<uint16_t*>(sf_dn + sf_tiled_offset(d, 2 * g32, K >> 4)) = dup;
    else sf_dn[sf_tiled_offset(d, g32, K >> 5)] = (uint8_t)bs.code;
  } else {
    sf_sp[d * (K >> 5) + g32] = (uint8_t)bs.code;
    if (FMT == SHARQ_NVFP4) *reinterpret_cast<uint16_t*>(sf_dn + d * (K >> 4) + 2 * g32) = dup;
    else sf_dn[d * (K >> 5) + g32] = (uint8_t)bs.code;
  }
}

cudaError_t launch_quantize_weight(const sharq_config* cfg, const void* W, int64_t D, int64_t K, int64_t ldw,
                                   void* codes, void* sf_sp, void* sf_dn, float* ts, void* workspace,
                                   cudaStream_t st) {
  uint32_t* amax = reinterpret_cast<uint32_t*>(workspace);
  cudaError_t e = cudaMemsetAsync(amax, 0, sizeof(uint32_t), st);
  if (e != cudaSuccess) return e;
  if (cfg->fmt == SHARQ_NVFP4) {
    weight_amax_kernel<<<1024, 256, 0, st>>>((const uint16_t*)W, D, K, ldw, amax);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  const int64_t items = D * ((K + 1023) >> 10);
  const unsigned blocks = (unsigned)((items * 32 + 255) / 256);
  const int tiled = cfg->layout == SHARQ_LAYOUT_TILED;
#define SHARQ_WQ(F) weight_quant_kernel<F><<<blocks, 256, 0, st>>>((const uint16_t*)W, D, K, ldw, (uint8_t*)codes, \
                                                                    (uint8_t*)sf_sp, (uint8_t*)sf_dn, ts, amax, tiled)
  if (cfg->fmt == SHARQ_NVFP4) SHARQ_WQ(SHARQ_NVFP4);
  else if (cfg->fmt == SHARQ_MXFP4) SHARQ_WQ(SHARQ_MXFP4);
  else SHARQ_WQ(SHARQ_HIF4);
#undef SHARQ_WQ
  return cudaGetLastError();
}

}  // namespace sharq
