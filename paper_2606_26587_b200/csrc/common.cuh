// Shared device helpers of the SharQ CUDA path (sm_100a only).  No host logic here.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/sharq.h"

namespace sharq {

// ---- tiled layouts (include/sharq.h "Output layouts") --------------------------------------
// scale factors: [rows, C] bytes, 512-byte atoms of 128 rows x 4 columns, atoms K-fastest.
__host__ __device__ __forceinline__ size_t sf_tiled_offset(int64_t r, int64_t c, int64_t C) {
  return (size_t)((r >> 7) * (C >> 2) + (c >> 2)) * 512 + (size_t)((r & 31) * 16 + ((r & 127) >> 5) * 4 + (c & 3));
}
// sparsity metadata: [rows, K/16] bytes, 2048-byte tiles of 128 rows x 16 bytes, K-fastest.
__host__ __device__ __forceinline__ size_t meta_tiled_offset(int64_t r, int64_t b, int64_t K) {
  return (size_t)((r >> 7) * (K >> 8) + (b >> 4)) * 2048 + (size_t)((r & 127) * 16 + (b & 15));
}
__host__ __device__ __forceinline__ int64_t round_up(int64_t a, int64_t b) { return (a + b - 1) / b * b; }

#ifdef __CUDACC__
// ---- small PTX wrappers ---------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ float bf16lo_to_f32(uint32_t packed) { return __uint_as_float(packed << 16); }
__device__ __forceinline__ float bf16hi_to_f32(uint32_t packed) { return __uint_as_float(packed & 0xFFFF0000u); }

// The same widenings on the FMA pipe (FHFMA.BF16: x * 1 + (-0), exact for every finite x and both zeros): sharq_prepare
// is bound by the ALU pipe (shifts, logic, min / max, conversions), the FMA pipe has room
__device__ __forceinline__ void bf16x2_to_f32_fma(uint32_t packed, float& lo, float& hi) {
#ifdef SHARQ_UNPACK_ALU
  lo = bf16lo_to_f32(packed); hi = bf16hi_to_f32(packed);
#else
  asm("{ .reg .b16 l, h, one;\n\t"
      "mov.b32 {l, h}, %2;\n\t"
      "mov.b16 one, 0x3F80;\n\t"
      "fma.rn.f32.bf16 %0, l, one, %3;\n\t"
      "fma.rn.f32.bf16 %1, h, one, %3; }"
      : "=f"(lo), "=f"(hi) : "r"(packed), "f"(-0.0f));
#endif
}

// fp32 pair -> packed bf16x2 (lo in the low half), round-to-nearest-even
__device__ __forceinline__ uint32_t pack_bf16x2_rn(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
// bf16x2 * bf16x2 -> bf16x2, one RNE rounding per half, subnormals kept
__device__ __forceinline__ uint32_t mul_bf16x2_rn(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}
__device__ __forceinline__ uint32_t add_bf16x2_rn(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("add.rn.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}
__device__ __forceinline__ uint32_t sub_bf16x2_rn(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("sub.rn.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}
// a * b + c per half: the exact product and sum, ONE RNE rounding to bf16
__device__ __forceinline__ uint32_t fma_bf16x2_rn(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t r;
  asm("fma.rn.bf16x2 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
  return r;
}
__device__ __forceinline__ uint32_t min_bf16x2(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("min.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}
__device__ __forceinline__ uint32_t abs_bf16x2(uint32_t a) {          // FMA pipe (a LOP3 would take an ALU slot)
  uint32_t r;
  asm("abs.bf16x2 %0, %1;" : "=r"(r) : "r"(a));
  return r;
}
// byte permute, integer multiply-add and (a & mask) | c as single instructions
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {   // only sel[15:0] is read
  uint32_t r;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(sel));
  return r;
}

__device__ __forceinline__ uint32_t mad_lo_u32(uint32_t a, uint32_t b, uint32_t c) {   // IMAD: FMA pipe
  uint32_t r;
  asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
  return r;
}
__device__ __forceinline__ uint32_t lop3_and_or(uint32_t a, uint32_t mask, uint32_t c) {   // (a & mask) | c
  uint32_t r;
  asm("lop3.b32 %0, %1, %2, %3, 0xF8;" : "=r"(r) : "r"(c), "r"(mask), "r"(a));
  return r;
}
// two fp32 -> one byte of two E2M1 codes (lo in the low nibble), RNE, saturating
__device__ __forceinline__ uint32_t cvt_e2m1x2(float lo, float hi) {
  uint32_t r;
  asm("{ .reg .b8 t; .reg .b16 h;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 t, %1, %2;\n\t"
      "mov.b16 h, {t, 0};\n\t"
      "cvt.u32.u16 %0, h; }"
      : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
// eight fp32 -> one word of eight E2M1 codes (element 0 in the low nibble), RNE, saturating
__device__ __forceinline__ uint32_t cvt_e2m1x8(float v0, float v1, float v2, float v3, float v4, float v5, float v6,
                                               float v7) {
  uint32_t r;
  asm("{ .reg .b8 t0, t1, t2, t3;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 t0, %2, %1;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 t1, %4, %3;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 t2, %6, %5;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 t3, %8, %7;\n\t"
      "mov.b32 %0, {t0, t1, t2, t3}; }"
      : "=r"(r) : "f"(v0), "f"(v1), "f"(v2), "f"(v3), "f"(v4), "f"(v5), "f"(v6), "f"(v7));
  return r;
}
// one byte of two E2M1 codes -> two fp32 values
__device__ __forceinline__ void e2m1x2_to_f32(uint32_t byte, float& lo, float& hi) {
  uint32_t h2;
  asm("{ .reg .b8 t, z; .reg .b16 h;\n\t"
      "cvt.u16.u32 h, %1;\n\t"
      "mov.b16 {t, z}, h;\n\t"
      "cvt.rn.f16x2.e2m1x2 %0, t; }"
      : "=r"(h2) : "r"(byte));
  __half2 v = *reinterpret_cast<__half2*>(&h2);
  float2 f = __half22float2(v);
  lo = f.x;
  hi = f.y;
}
// non-negative fp32 -> E4M3 code, RNE, saturating at 448
__device__ __forceinline__ uint32_t cvt_e4m3(float x) {
  uint16_t r;
  asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(0.0f), "f"(x));
  return (uint32_t)(r & 0xFF);
}
__device__ __forceinline__ float e4m3_to_f32(uint32_t code) {
  uint32_t h2;
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"((uint16_t)code));
  return __half2float(__ushort_as_half((unsigned short)(h2 & 0xFFFF)));
}
// non-negative fp32 -> E8M0 code e+127, 2^e the smallest power of two >= x, e clamped to [-127,127]
__device__ __forceinline__ uint32_t e8m0_round_up(float x) {
  uint32_t b = __float_as_uint(x), e = b >> 23, m = b & 0x7FFFFFu;
  uint32_t code = (e == 0) ? (m > 0x400000u ? 1u : 0u) : e + (m != 0u ? 1u : 0u);
  return code > 254u ? 254u : code;
}
__device__ __forceinline__ float e8m0_to_f32(uint32_t code) {
  return __uint_as_float(code == 0 ? 0x00400000u : code << 23);
}
__device__ __forceinline__ float e8m0_inv_to_f32(uint32_t code) {  // 2^(127-code)
  return __uint_as_float(code == 254u ? 0x00400000u : (254u - code) << 23);
}
#endif  // __CUDACC__

}  // namespace sharq
