// sharq_linear for HiF4.
//
// B200's tcgen05 has no S1P2 element / E6M2 scale format, so HiF4 has no FP4-rate tensor path.  Every
// HiF4 value E6M2 * 2^(E1_8 + E1_16) * S1P2 = (4 + m) * k * 2^(E - 52 + shift) with (4 + m) * k <= 49
// has at most 6 significant bits, i.e. it is EXACT in bf16.  The path is therefore:
//   1. weights: bf16 [D, K] ONCE, by sharq_quantize_weight (the HiF4 "dense view" of the payload is this bf16 tensor);
//   2. activations, per call (hif4_dequant_act_sparse_kernel): backbone compressed [T, K/2] bf16 + 2:4 metadata in the
//      tensor core's tiling, residual [T, K] bf16;
//   3. hif4_gemm_sp_pair_kernel: CTA-pair tiles, tcgen05.mma.sp kind::f16 on the backbone, dense tcgen05.mma kind::f16
//      on the residual, one fp32 accumulator: Y = A_sp W^T + A_dn W^T.
// Small launches keep the first version: activations as [T, 2K] = [backbone with zeros | residual] and a dense bf16
// GEMM over the 2K-long rows (hif4_gemm_kernel).
// Roofline denominator: the measured bf16 tensor peak.
#include <cuda.h>
#include <cuda_runtime.h>

#include <atomic>

#include "common.cuh"
#include "linear_args.h"
#include "tc_ptx.cuh"
#include "epilogue.cuh"

namespace sharq {

namespace {

// bf16 bits of one decoded HiF4 element (Eq. 15): code = S1P2 nibble, word = E6M2 | E1_8<<8 | E1_16<<16,
// i = position inside the 64-element unit.
__device__ __forceinline__ uint32_t hif4_to_bf16(uint32_t code, uint32_t word, uint32_t i) {
  const uint32_t k = code & 7u;
  const uint32_t n = (4u + (word & 3u)) * k;                               // <= 49: exact
  const int shift = (int)((word >> (8 + (i >> 3))) & 1u) + (int)((word >> (16 + (i >> 2))) & 1u);
  const int p = (int)((word >> 2) & 63u) - 52 + shift;                     // value = n * 2^p
  const float v = __fmul_rn((float)n, __uint_as_float((uint32_t)(p + 127) << 23));
  return (__float_as_uint(v) >> 16) | ((code & 8u) << 12);                 // exact in bf16; sign of the code
}

// activations: one thread per 8 logical k (two 2:4 groups)
__global__ void hif4_dequant_act_kernel(const uint8_t* __restrict__ sp_codes, const uint32_t* __restrict__ sp_sf,
                                        const uint8_t* __restrict__ sp_meta, const uint8_t* __restrict__ dn_codes,
                                        const uint32_t* __restrict__ dn_sf, uint16_t* __restrict__ A, int64_t T,
                                        int64_t K, int path) {
  tc::grid_dependency_wait();
  const int64_t n8 = K >> 3;
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < T * n8;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int64_t t = idx / n8, c = idx % n8;          // k = 8c .. 8c+7
    const uint32_t unit_i = (uint32_t)((8 * c) & 63);
    uint32_t sp[8], dn[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) sp[i] = 0u, dn[i] = 0u;
    if (path != 2) {
      const uint32_t word = sp_sf[t * (K >> 6) + (c >> 3)];
      const uint32_t meta = sp_meta[t * (K >> 3) + c];                 // two nibbles: groups 2c, 2c+1
      const uint32_t codes = *reinterpret_cast<const uint16_t*>(sp_codes + t * (K >> 2) + 2 * c);
#pragma unroll
      for (int g = 0; g < 2; ++g) {
        const uint32_t nib = (meta >> (4 * g)) & 15u, i0 = nib & 3u, i1 = nib >> 2;
        const uint32_t byte = (codes >> (8 * g)) & 255u;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          uint32_t v = 0u;
          if ((uint32_t)e == i0) v = hif4_to_bf16(byte & 15u, word, unit_i + 4 * g + e);
          if ((uint32_t)e == i1) v = hif4_to_bf16(byte >> 4, word, unit_i + 4 * g + e);
          sp[4 * g + e] = v;
        }
      }
    }
    if (path != 1) {
      const uint32_t word = dn_sf[t * (K >> 6) + (c >> 3)];
      const uint32_t codes = *reinterpret_cast<const uint32_t*>(dn_codes + t * (K >> 1) + 4 * c);
#pragma unroll
      for (int e = 0; e < 8; ++e) dn[e] = hif4_to_bf16((codes >> (4 * e)) & 15u, word, unit_i + e);
    }
    uint16_t* row = A + t * (2 * K);
    *reinterpret_cast<uint4*>(row + 8 * c) =
        make_uint4(sp[0] | sp[1] << 16, sp[2] | sp[3] << 16, sp[4] | sp[5] << 16, sp[6] | sp[7] << 16);
    *reinterpret_cast<uint4*>(row + K + 8 * c) =
        make_uint4(dn[0] | dn[1] << 16, dn[2] | dn[3] << 16, dn[4] | dn[5] << 16, dn[6] | dn[7] << 16);
  }
}

__global__ void hif4_dequant_weight_kernel(const uint8_t* __restrict__ codes, const uint32_t* __restrict__ sf,
                                           uint16_t* __restrict__ W, int64_t D, int64_t K) {
  const int64_t n8 = K >> 3;
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < D * n8;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int64_t d = idx / n8, c = idx % n8;
    const uint32_t word = sf[d * (K >> 6) + (c >> 3)];
    const uint32_t cw = *reinterpret_cast<const uint32_t*>(codes + d * (K >> 1) + 4 * c);
    uint32_t v[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) v[e] = hif4_to_bf16((cw >> (4 * e)) & 15u, word, (uint32_t)((8 * c) & 63) + e);
    *reinterpret_cast<uint4*>(W + d * K + 8 * c) =
        make_uint4(v[0] | v[1] << 16, v[2] | v[3] << 16, v[4] | v[5] << 16, v[6] | v[7] << 16);
  }
}

// ---- dense bf16 GEMM: Y[T, D] = A[T, 2K] * [W | W]^T, 128 x BN tiles, persistent, 2 TMEM accumulators ---
constexpr int GM = 128, GK = 64, kGemmThreads = 192;

struct GemmParams {
  const float *row_scale, *w_ts;
  const uint16_t* bias;
  void* Y;
  int64_t ldy;
  int32_t T, D, K, out_fp32, m_blocks, total_tiles;
  int32_t group_m;     // pair kernel: 256-row blocks per supertile (epilogue.cuh pair_tile)
};

__device__ __forceinline__ uint32_t idesc_bf16(uint32_t M, uint32_t N) {
  return (1u << 4) /*fp32 accumulate*/ | (1u << 7) /*A bf16*/ | (1u << 10) /*B bf16*/ | ((N >> 3) << 17) |
         ((M >> 4) << 24);
}
__device__ __forceinline__ void mma_bf16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                         uint32_t accumulate) {
  asm volatile("{ .reg .pred p;\n\t"
               "setp.ne.b32 p, %4, 0;\n\t"
               "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p; }"
               ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}

template <int BN>
__global__ void __launch_bounds__(kGemmThreads, 1)
hif4_gemm_kernel(const __grid_constant__ CUtensorMap tm_a, const __grid_constant__ CUtensorMap tm_w,
                 const GemmParams p) {
  constexpr int A_BYTES = GM * 128, B_BYTES = BN * 128, STAGE = A_BYTES + B_BYTES;
  constexpr int STAGES = (BN == 256) ? 4 : 6;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bars = smem_base + STAGES * STAGE;
  auto full_bar = [&](int s) { return bars + 8u * s; };
  auto empty_bar = [&](int s) { return bars + 8u * (STAGES + s); };
  auto tmem_full_bar = [&](int a) { return bars + 8u * (2 * STAGES + a); };
  auto tmem_empty_bar = [&](int a) { return bars + 8u * (2 * STAGES + 2 + a); };
  const uint32_t tmem_ptr_smem = bars + 8u * (2 * STAGES + 4);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int num_kb = 2 * p.K / GK, half_kb = p.K / GK;

  if (warp == 0 && lane == 0) {
    tc::prefetch_tmap(&tm_a);
    tc::prefetch_tmap(&tm_w);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) {
      tc::mbar_init(full_bar(s), 1);
      tc::mbar_init(empty_bar(s), 1);
    }
    for (int a = 0; a < 2; ++a) {
      tc::mbar_init(tmem_full_bar(a), 1);
      tc::mbar_init(tmem_empty_bar(a), 4);
    }
    tc::fence_mbar_init();
  }
  if (warp == 2) tc::tmem_alloc<512>(tmem_ptr_smem);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_smem));
  tc::grid_dependency_wait();                            // A / W were dequantised by the kernels before us

  if (warp == 0) {
    const bool lead = tc::elect_one() != 0;
    const uint64_t pol = tc::policy_evict_normal();
    uint32_t it = 0;
    for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x) {
      const int m_blk = tile % p.m_blocks, n_blk = tile / p.m_blocks;
      for (int kb = 0; kb < num_kb; ++kb, ++it) {
        const int s = it % STAGES;
        tc::mbar_wait(empty_bar(s), ((it / STAGES) & 1) ^ 1);
        const uint32_t st = smem_base + s * STAGE;
        if (lead) tc::mbar_expect_tx(full_bar(s), STAGE);
        if (lead) tc::tma_load_2d(st, &tm_a, full_bar(s), kb * GK, m_blk * GM, pol);
        if (lead) tc::tma_load_2d(st + A_BYTES, &tm_w, full_bar(s), (kb % half_kb) * GK, n_blk * BN, pol);
      }
    }
  } else if (warp == 1) {
    const bool lead = tc::elect_one() != 0;
    const uint32_t idesc = idesc_bf16(GM, BN);
    uint32_t it = 0, n_unit = 0;
    for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x, ++n_unit) {
      const uint32_t as = n_unit & 1u;
      tc::mbar_wait(tmem_empty_bar(as), ((n_unit >> 1) & 1u) ^ 1u);
      tc::tc_fence_after();
      uint32_t accumulate = 0;
      for (int kb = 0; kb < num_kb; ++kb, ++it) {
        const int s = it % STAGES;
        tc::mbar_wait(full_bar(s), (it / STAGES) & 1);
        tc::tc_fence_after();
        const uint32_t st = smem_base + s * STAGE;
#pragma unroll
        for (int j = 0; j < GK / 16; ++j) {              // UMMA K = 16 bf16 = 32 bytes
          if (lead) mma_bf16(tmem_base + as * BN, tc::smem_desc(st + 32 * j, 1024, 2),
                             tc::smem_desc(st + A_BYTES + 32 * j, 1024, 2), idesc, accumulate);
          accumulate = 1;
        }
        if (lead) tc::tc_commit(empty_bar(s));
      }
      if (lead) tc::tc_commit(tmem_full_bar(as));
    }
  } else {
    const int sub = warp & 3, r_local = sub * 32 + lane;
    const uint32_t lane_addr = tmem_base + ((uint32_t)(sub * 32) << 16);
    uint32_t n_unit = 0;
    for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x, ++n_unit) {
      const int m_blk = tile % p.m_blocks, n_blk = tile / p.m_blocks;
      const uint32_t as = n_unit & 1u;
      const int64_t row = (int64_t)m_blk * GM + r_local;
      const bool row_ok = row < p.T;
      const float scale = row_ok ? __fmul_rn(p.row_scale[row], p.w_ts[0]) : 0.0f;
      tc::mbar_wait(tmem_full_bar(as), (n_unit >> 1) & 1u);
      tc::tc_fence_after();
#pragma unroll 1
      for (int c = 0; c < BN / 32; ++c) {
        uint32_t v[32];
        tc::tmem_ld32(lane_addr + as * BN + c * 32, v);
        tc::tmem_ld_wait();
        if (row_ok) {
          const int col0 = n_blk * BN + c * 32;
          float f[32];
#pragma unroll
          for (int i = 0; i < 32; ++i) f[i] = __fmul_rn(__uint_as_float(v[i]), scale);
          if (p.bias) {
#pragma unroll
            for (int i = 0; i < 32; ++i) f[i] = __fadd_rn(f[i], __uint_as_float((uint32_t)p.bias[col0 + i] << 16));
          }
          if (p.out_fp32) {
            float4* dst = reinterpret_cast<float4*>(static_cast<float*>(p.Y) + row * p.ldy + col0);
#pragma unroll
            for (int i = 0; i < 8; ++i) dst[i] = make_float4(f[4 * i], f[4 * i + 1], f[4 * i + 2], f[4 * i + 3]);
          } else {
            uint4* dst = reinterpret_cast<uint4*>(static_cast<uint16_t*>(p.Y) + row * p.ldy + col0);
#pragma unroll
            for (int i = 0; i < 4; ++i)
              dst[i] = make_uint4(pack_bf16x2_rn(f[8 * i], f[8 * i + 1]), pack_bf16x2_rn(f[8 * i + 2], f[8 * i + 3]),
                                  pack_bf16x2_rn(f[8 * i + 4], f[8 * i + 5]), pack_bf16x2_rn(f[8 * i + 6], f[8 * i + 7]));
          }
        }
      }
      tc::tc_fence_before();
      __syncwarp();
      if (lane == 0) tc::mbar_arrive(tmem_empty_bar(as));
    }
  }
  __syncthreads();
  if (warp == 2) {
    tc::tc_fence_after();
    tc::tmem_dealloc<512>(tmem_base);
  }
}

// ---- CTA-pair MMAs (cta_group::2): each CTA stages its own 128 rows of A and HALF of the W tile, one tcgen05.mma of
// M = 256 consumes both CTAs' shared memory --------------------------------------------------------------------
__device__ __forceinline__ void mma_bf16_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                              uint32_t accumulate) {
  asm volatile("{ .reg .pred p;\n\t"
               "setp.ne.b32 p, %4, 0;\n\t"
               "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p; }"
               ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}

// ---- 2:4-sparse backbone: tcgen05.mma.sp kind::f16 (SURVEY.md 8(a) S12 as written) --------------------------------
// The backbone half of a HiF4 activation is 2:4 sparse by construction: instead of multiplying a dense
// [T, K] bf16 matrix with explicit zeros, the survivors go in compressed, [T, K/2] bf16 in ascending k (exactly the order
// of sp_codes), and the 2-bit indices of sharq_prepare's metadata nibbles (i0 | i1 << 2 per 4 elements) tell the
// tensor core where they belong: half the A bytes and half the MMA time of the dense emulation for that half.
// Metadata layout the sparse bf16 MMA expects (CUTLASS sm1xx_sparse_config.inl, TensorEAtom_MMA_F16, used as a hardware
// spec): one 2048-byte atom per 128 rows x 128 logical k; byte of (row m, logical k) inside the atom =
//   16 (m % 8) + 2 ((m / 8) % 2) + 256 (m / 16) + 128 ((k / 16) % 2) + 4 (k / 32) + (k % 16) / 8,
// so that one tcgen05.cp.128x128b puts the four 32-bit columns of the four K = 32 MMAs of the atom into tensor memory.
//
// The decode itself is packed bf16x2 (the values are exact in bf16): value = m qup, m the 3 magnitude bits of the code,
// qup = 0.25 * E6M2 * 2^(E1_8 + E1_16) a bf16 number whose bits are the E6M2 code shifted into place plus exponent-field
// offsets.  The code nibbles of two neighbouring elements go into the low mantissa bits of 128.0 (0x4300 | m per half),
// one fma.rn.bf16x2 (128 + m) qup - 128 qup gives m qup exactly, the sign nibble bits are OR-ed in.
struct Hif4Qup { uint32_t qa, nqa, qb, nqb; };   // qup and -128 qup (bf16x2 splats) of the thread's two 4-groups

// `word` = E6M2 | E1_8 << 8 | E1_16 << 16 of the unit, g8 = index of the thread's 8 elements inside the 64-element unit
__device__ __forceinline__ Hif4Qup hif4_qup(uint32_t word, uint32_t g8) {
  const uint32_t base = ((word & 0xFFu) << 5) + (79u << 7) - 0x100u;        // bf16 bits of 0.25 * E6M2 (R11: bias 48)
  const uint32_t e8 = (word >> (8 + g8)) & 1u, e16 = (word >> (16 + 2 * g8)) & 3u;
  Hif4Qup q;
  q.qa = (base + ((e8 + (e16 & 1u)) << 7)) * 0x10001u;
  q.qb = (base + ((e8 + (e16 >> 1)) << 7)) * 0x10001u;
  q.nqa = q.qa + 0x83808380u;                                                // exponent + 7, sign set: no carry between halves
  q.nqb = q.qb + 0x83808380u;
  return q;
}

// elements 2j, 2j + 1 of a word of code nibbles (ascending k) -> bf16x2
__device__ __forceinline__ uint32_t hif4_decode2(uint32_t L, uint32_t H, uint32_t Se, uint32_t So, int j, uint32_t q,
                                                 uint32_t nq) {
  const uint32_t sel = 0x4400u + 0x1111u * (uint32_t)j;                      // bytes [lo_j, lo_j, hi_j, hi_j]
  const uint32_t tq = lop3_and_or(prmt(L, H, sel), 0x00FF00FFu, 0x43004300u);
  return lop3_and_or(prmt(Se, So, sel), 0x80008000u, fma_bf16x2_rn(tq, q, nq));
}

// grid: x over the K / 8 element groups of a row (one thread each), y over blocks of kDqRows consecutive rows: the
// thread keeps its column-derived offsets and walks down the rows with pointer increments
constexpr int kDqRows = 8;                             // Tp is a multiple of 128

__global__ void __launch_bounds__(128)
hif4_dequant_act_sparse_kernel(const uint8_t* __restrict__ sp_codes, const uint32_t* __restrict__ sp_sf,
                               const uint8_t* __restrict__ sp_meta, const uint8_t* __restrict__ dn_codes,
                               const uint32_t* __restrict__ dn_sf, uint16_t* __restrict__ Asp,
                               uint16_t* __restrict__ Adn, uint8_t* __restrict__ E, int64_t T, int64_t Tp,
                               int64_t K, int path) {
  tc::grid_dependency_wait();
  const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;                  // k = 8c .. 8c + 7: one E1_8 group
  if (c >= (uint32_t)(K >> 3)) return;
  const uint32_t g8 = c & 7u, kk = (8u * c) & 127u;
  for (int64_t t0 = (int64_t)blockIdx.y * kDqRows; t0 < Tp; t0 += (int64_t)gridDim.y * kDqRows) {
  // row-invariant offsets; all rows of the block lie in one 128-row metadata atom row (kDqRows divides 128)
  const uint8_t* p_meta = sp_meta + t0 * (K >> 3) + c;
  const uint32_t* p_spsf = sp_sf + t0 * (K >> 6) + (c >> 3);
  const uint32_t* p_dnsf = dn_sf + t0 * (K >> 6) + (c >> 3);
  const uint8_t* p_spc = sp_codes + t0 * (K >> 2) + 2 * c;
  const uint8_t* p_dnc = dn_codes + t0 * (K >> 1) + 4 * c;
  uint16_t* p_asp = Asp + t0 * (K >> 1) + 4 * c;
  uint16_t* p_adn = Adn + t0 * K + 8 * c;
  uint8_t* p_e = E + ((t0 >> 7) * (K >> 7) + (c >> 4)) * 2048 + 128u * ((kk >> 4) & 1u) + 4u * (kk >> 5) + ((kk & 15u) >> 3);
  const int64_t rows_valid = T - t0;                   // rows >= T are pad rows: a valid nibble, zero values
#pragma unroll 4
  for (int i = 0; i < kDqRows; ++i) {
    uint2 sp = make_uint2(0u, 0u);
    uint4 dn = make_uint4(0u, 0u, 0u, 0u);
    uint32_t meta = 0x44u;
    if (i < rows_valid) {
      meta = p_meta[(int64_t)i * (K >> 3)];            // two nibbles: 4-groups 2c, 2c+1
      if (path != 2) {
        const Hif4Qup q = hif4_qup(p_spsf[(int64_t)i * (K >> 6)], g8);
        // two bytes: the survivors i0 < i1 of each 4-group, ascending k, exactly the compressed operand's order
        const uint32_t codes = *reinterpret_cast<const uint16_t*>(p_spc + (int64_t)i * (K >> 2));
        const uint32_t L = codes & 0x0707u, H = (codes >> 4) & 0x0707u, Se = (codes << 4) & 0x8080u, So = codes & 0x8080u;
        sp.x = hif4_decode2(L, H, Se, So, 0, q.qa, q.nqa);
        sp.y = hif4_decode2(L, H, Se, So, 1, q.qb, q.nqb);
      }
      if (path != 1) {
        const Hif4Qup q = hif4_qup(p_dnsf[(int64_t)i * (K >> 6)], g8);
        const uint32_t codes = *reinterpret_cast<const uint32_t*>(p_dnc + (int64_t)i * (K >> 1));
        const uint32_t L = codes & 0x07070707u, H = (codes >> 4) & 0x07070707u;
        const uint32_t Se = (codes << 4) & 0x80808080u, So = codes & 0x80808080u;
        dn.x = hif4_decode2(L, H, Se, So, 0, q.qa, q.nqa);
        dn.y = hif4_decode2(L, H, Se, So, 1, q.qa, q.nqa);
        dn.z = hif4_decode2(L, H, Se, So, 2, q.qb, q.nqb);
        dn.w = hif4_decode2(L, H, Se, So, 3, q.qb, q.nqb);
      }
    }
    *reinterpret_cast<uint2*>(p_asp + (int64_t)i * (K >> 1)) = sp;
    *reinterpret_cast<uint4*>(p_adn + (int64_t)i * K) = dn;
    const uint32_t m = ((uint32_t)t0 + (uint32_t)i) & 127u;
    p_e[16 * (m & 7) + 2 * ((m >> 3) & 1) + 256 * (m >> 4)] = (uint8_t)meta;
  }
  }
}

__device__ __forceinline__ void mma_bf16_sparse_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                                     uint32_t meta_tmem, uint32_t accumulate) {
  asm volatile("{ .reg .pred p;\n\t"
               "setp.ne.b32 p, %4, 0;\n\t"
               "tcgen05.mma.sp.cta_group::2.kind::f16 [%0], %1, %2, [%5], %3, p; }"
               ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate), "r"(meta_tmem) : "memory");
}

// One pipeline stage = 128 logical k.  Sparse step: A_sp 128 rows x 64 stored bf16 (16 KB) + metadata atom (2 KB) + this
// CTA's half of the W tile as two 64-k sub-tiles; dense step: two A sub-tiles (32 KB) + the same W bytes.
template <int BN>
struct SpStage {
  static constexpr int HALF = BN / 2;
  static constexpr int A0 = 0, A1 = 16384, META = 16384, B0 = 32768, B1 = B0 + HALF * 128;
  static constexpr int BYTES = (B1 + HALF * 128 + 1023) / 1024 * 1024;
  static constexpr int STAGES = 3;
  static constexpr int E_COL = 2 * BN;                     // two accumulator stages, then four metadata columns
  static constexpr int SMEM = STAGES * BYTES + 1024 + 256 + kStageBytes;
  static_assert(E_COL + 4 <= 512, "tensor memory");
};

template <int BN>
__global__ void __launch_bounds__(kGemmThreads, 1)
hif4_gemm_sp_pair_kernel(const __grid_constant__ CUtensorMap tm_asp, const __grid_constant__ CUtensorMap tm_adn,
                         const __grid_constant__ CUtensorMap tm_w, const __grid_constant__ CUtensorMap tm_e,
                         const GemmParams p, const int path) {
  using S = SpStage<BN>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bars = smem_base + S::STAGES * S::BYTES;
  auto full_bar = [&](int s) { return bars + 8u * s; };                       // leader CTA
  auto empty_bar = [&](int s) { return bars + 8u * (S::STAGES + s); };
  auto tmem_full_bar = [&](int a) { return bars + 8u * (2 * S::STAGES + a); };
  auto tmem_empty_bar = [&](int a) { return bars + 8u * (2 * S::STAGES + 2 + a); };   // leader CTA
  const uint32_t tmem_ptr_smem = bars + 8u * (2 * S::STAGES + 4);
  const uint32_t stg_base = bars + 256u;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rank = (int)tc::cluster_ctarank();
  const int ksteps = p.K / 128;                                    // per phase
  const int sp_steps = path != 2 ? ksteps : 0, dn_steps = path != 1 ? ksteps : 0;
  const int m_pairs = (p.m_blocks + 1) / 2, n_tiles = (p.D + BN - 1) / BN, total = m_pairs * n_tiles;
  const int gm = p.group_m > 0 && p.group_m < m_pairs ? p.group_m : m_pairs;
  const int tile0 = (int)tc::cluster_id_x(), tile_step = (int)(gridDim.x >> 1);

  if (warp == 0 && lane == 0) {
    tc::prefetch_tmap(&tm_asp);
    tc::prefetch_tmap(&tm_adn);
    tc::prefetch_tmap(&tm_w);
    tc::prefetch_tmap(&tm_e);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < S::STAGES; ++s) {
      tc::mbar_init(full_bar(s), 1);
      tc::mbar_init(empty_bar(s), 1);
    }
    for (int a = 0; a < 2; ++a) {
      tc::mbar_init(tmem_full_bar(a), 1);
      tc::mbar_init(tmem_empty_bar(a), 8);
    }
    tc::fence_mbar_init();
  }
  if (warp == 2) tc::tmem_alloc_pair<512>(tmem_ptr_smem);
  tc::tc_fence_before();
  __syncwarp();
  tc::cluster_sync_all();
  tc::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_smem));
  tc::grid_dependency_wait();

  if (warp == 0) {
    const bool lead = tc::elect_one() != 0;
    const uint64_t pol = tc::policy_evict_normal();
    const uint32_t w_bytes = 2u * S::HALF * 128u;
    uint32_t it = 0;
    for (int tile = tile0; tile < total; tile += tile_step) {
      int m_pair, n_blk;
      pair_tile(tile, m_pairs, n_tiles, gm, m_pair, n_blk);
      const int m_blk = 2 * m_pair + rank;
      const int m_e = min(m_blk, p.m_blocks - 1);                  // a ragged pair's second CTA: valid memory, unused rows
      const int w_row = n_blk * BN + rank * S::HALF;
      for (int ks = 0; ks < sp_steps + dn_steps; ++ks, ++it) {
        const int s = it % S::STAGES;
        tc::mbar_wait(empty_bar(s), ((it / S::STAGES) & 1) ^ 1);
        const uint32_t st = smem_base + s * S::BYTES;
        const uint32_t fb = full_bar(s);
        const bool sparse = ks < sp_steps;
        const int k128 = sparse ? ks : ks - sp_steps;
        if (lead && rank == 0) tc::mbar_expect_tx(fb, 2u * (w_bytes + (sparse ? 16384u + 2048u : 32768u)));
        if (lead) tc::tma_load_2d_pair(st + S::B0, &tm_w, fb, k128 * 128, w_row, pol);
        if (lead) tc::tma_load_2d_pair(st + S::B1, &tm_w, fb, k128 * 128 + 64, w_row, pol);
        if (sparse) {
          if (lead) tc::tma_load_2d_pair(st + S::A0, &tm_asp, fb, k128 * 64, m_blk * GM, pol);
          if (lead) tc::tma_load_2d_pair(st + S::META, &tm_e, fb, 0, (m_e * ksteps + k128) * 2, pol);
        } else {
          if (lead) tc::tma_load_2d_pair(st + S::A0, &tm_adn, fb, k128 * 128, m_blk * GM, pol);
          if (lead) tc::tma_load_2d_pair(st + S::A1, &tm_adn, fb, k128 * 128 + 64, m_blk * GM, pol);
        }
      }
    }
  } else if (warp == 1) {
    if (rank == 0) {
      const bool lead = tc::elect_one() != 0;
      const uint32_t idesc = idesc_bf16(256, BN), idesc_sp = idesc | (1u << 2);
      uint32_t it = 0, n_unit = 0;
      for (int tile = tile0; tile < total; tile += tile_step, ++n_unit) {
        const uint32_t as = n_unit & 1u;
        const uint32_t acc = tmem_base + as * BN;
        tc::mbar_wait(tmem_empty_bar(as), ((n_unit >> 1) & 1u) ^ 1u);
        tc::tc_fence_after();
        uint32_t accumulate = 0;
        for (int ks = 0; ks < sp_steps + dn_steps; ++ks, ++it) {
          const int s = it % S::STAGES;
          tc::mbar_wait(full_bar(s), (it / S::STAGES) & 1);
          tc::tc_fence_after();
          const uint32_t st = smem_base + s * S::BYTES;
          if (ks < sp_steps) {
            if (lead) tc::tc_cp_meta_pair(tmem_base + S::E_COL, tc::smem_desc(st + S::META, 128, 0));
#pragma unroll
            for (int j = 0; j < 4; ++j) {                  // K = 32 logical = 16 stored bf16 (32 bytes of A) per MMA
              // the metadata address is an EVEN tensor-memory column; bit 0 of the instruction descriptor ("sparse id")
              // selects the even or the odd column of the pair
              if (lead) mma_bf16_sparse_pair(acc, tc::smem_desc(st + S::A0 + 32 * j, 1024, 2),
                                             tc::smem_desc(st + (j < 2 ? S::B0 : S::B1) + 64 * (j & 1), 1024, 2),
                                             idesc_sp | (uint32_t)(j & 1), tmem_base + S::E_COL + (j & ~1), accumulate);
              accumulate = 1;
            }
          } else {
#pragma unroll
            for (int j = 0; j < 8; ++j) {                  // K = 16 per MMA
              if (lead) mma_bf16_pair(acc, tc::smem_desc(st + (j < 4 ? S::A0 : S::A1) + 32 * (j & 3), 1024, 2),
                                      tc::smem_desc(st + (j < 4 ? S::B0 : S::B1) + 32 * (j & 3), 1024, 2), idesc, accumulate);
              accumulate = 1;
            }
          }
          if (lead) tc::tc_commit_pair(empty_bar(s), 3);
        }
        if (lead) tc::tc_commit_pair(tmem_full_bar(as), 3);
      }
    }
  } else {
    const int sub = warp & 3, r_local = sub * 32 + lane;
    const uint32_t lane_addr = tmem_base + ((uint32_t)(sub * 32) << 16);
    uint32_t n_unit = 0;
    for (int tile = tile0; tile < total; tile += tile_step, ++n_unit) {
      int m_pair, n_blk;
      pair_tile(tile, m_pairs, n_tiles, gm, m_pair, n_blk);
      const int m_blk = 2 * m_pair + rank;
      const uint32_t as = n_unit & 1u;
      const int64_t row = (int64_t)m_blk * GM + r_local;
      const float scale = row < p.T ? __fmul_rn(p.row_scale[row], p.w_ts[0]) : 0.0f;
      tc::mbar_wait(tmem_full_bar(as), (n_unit >> 1) & 1u);
      tc::tc_fence_after();
      const int rows_ok = (int)min((int64_t)32, max((int64_t)0, (int64_t)p.T - ((int64_t)m_blk * GM + sub * 32)));
      epilogue_tile<BN>(p, lane_addr + as * BN, stg_base + (uint32_t)sub * 4096u, lane, (int64_t)m_blk * GM + sub * 32, rows_ok,
                        n_blk * BN, scale);
      tc::tc_fence_before();
      __syncwarp();
      if (lane == 0) tc::mbar_arrive_cluster(tc::map_to_cta(tmem_empty_bar(as), 0));
    }
  }
  tc::tc_fence_before();
  __syncwarp();
  tc::cluster_sync_all();
  if (warp == 2) {
    tc::tc_fence_after();
    tc::tmem_dealloc_pair<512>(tmem_base);
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

bool make_bf16_map(CUtensorMap* m, const void* base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
  static EncodeTiledFn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      f = nullptr;
    return reinterpret_cast<EncodeTiledFn>(f);
  }();
  if (!fn) return false;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {cols * 2};
  cuuint32_t box[2] = {GK, box_rows};
  cuuint32_t estr[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int BN>
sharq_status launch_gemm(const CUtensorMap& tm_a, const CUtensorMap& tm_w, const GemmParams& p, int num_sms,
                         cudaStream_t st) {
  constexpr int STAGES = (BN == 256) ? 4 : 6;
  constexpr int SMEM = STAGES * (GM * 128 + BN * 128) + 1024 + 256;
  auto kfn = hif4_gemm_kernel<BN>;
  if (cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM) != cudaSuccess) return SHARQ_ECUDA;
  const int grid = p.total_tiles < num_sms ? p.total_tiles : num_sms;
  kfn<<<grid, kGemmThreads, SMEM, st>>>(tm_a, tm_w, p);
  return cudaGetLastError() == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}

}  // namespace

size_t hif4_linear_workspace_bytes(int64_t T, int64_t, int64_t K) {
  const int64_t Tp = round_up(T, 128);
  return (size_t)Tp * (size_t)(2 * K) * 2 + 256;       // the bf16 copy of the activation operands [T, 2K]
}

// offline, once per weight (sharq_quantize_weight): the bf16 view of the HiF4 payload
cudaError_t launch_hif4_dequant_weight(const void* codes, const void* sf, void* W_bf16, int64_t D, int64_t K,
                                       cudaStream_t st) {
  const int64_t nw = D * (K >> 3);
  if (nw == 0) return cudaSuccess;
  hif4_dequant_weight_kernel<<<(unsigned)((nw + 255) / 256 < 16384 ? (nw + 255) / 256 : 16384), 256, 0, st>>>(
      (const uint8_t*)codes, (const uint32_t*)sf, (uint16_t*)W_bf16, D, K);
  return cudaGetLastError();
}

namespace {
// [rows1k][256 u32] view of a byte buffer, boxes of `box_rows` 1024-byte rows (the metadata atoms: 2 rows each)
bool make_rows1k_map(CUtensorMap* m, const void* base, uint64_t bytes, uint32_t box_rows) {
  void* f = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
      q != cudaDriverEntryPointSuccess || bytes % 1024 != 0)
    return false;
  cuuint64_t dims[2] = {256, bytes / 1024};
  cuuint64_t strides[1] = {1024};
  cuuint32_t box[2] = {256, box_rows};
  cuuint32_t estr[2] = {1, 1};
  return reinterpret_cast<EncodeTiledFn>(f)(m, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, const_cast<void*>(base), dims, strides, box, estr,
                                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int BN>
sharq_status launch_sp_pair(const LinearArgs& a, void* workspace, int64_t Tp, int64_t m_blocks, int num_sms, cudaStream_t st) {
  using S = SpStage<BN>;
  // workspace: A_sp bf16 [Tp, K/2] | A_dn bf16 [Tp, K] | metadata atoms [Tp/128][K/128][2048]  (3.125 Tp K bytes of the 4 Tp K)
  uint8_t* base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(workspace) + 127) & ~(uintptr_t)127);
  uint16_t* Asp = reinterpret_cast<uint16_t*>(base);
  uint16_t* Adn = reinterpret_cast<uint16_t*>(base + (size_t)Tp * (size_t)a.K);
  uint8_t* E = base + (size_t)Tp * (size_t)a.K * 3;
  const uint16_t* W = reinterpret_cast<const uint16_t*>(a.w_sf_dn);
  const dim3 dq_grid((unsigned)(((a.K >> 3) + 127) / 128), (unsigned)(Tp / kDqRows < 65535 ? Tp / kDqRows : 65535));
  hif4_dequant_act_sparse_kernel<<<dq_grid, 128, 0, st>>>(
      (const uint8_t*)a.sp_codes, (const uint32_t*)a.sp_sf, (const uint8_t*)a.sp_meta, (const uint8_t*)a.dn_codes,
      (const uint32_t*)a.dn_sf, Asp, Adn, E, a.T, Tp, a.K, a.path);
  if (cudaGetLastError() != cudaSuccess) return SHARQ_ECUDA;
  CUtensorMap tm_asp, tm_adn, tm_w, tm_e;
  if (!make_bf16_map(&tm_asp, Asp, (uint64_t)Tp, (uint64_t)(a.K / 2), GM) ||
      !make_bf16_map(&tm_adn, Adn, (uint64_t)Tp, (uint64_t)a.K, GM) ||
      !make_bf16_map(&tm_w, W, (uint64_t)a.D, (uint64_t)a.K, S::HALF) ||
      !make_rows1k_map(&tm_e, E, (uint64_t)Tp * (uint64_t)a.K / 8, 2))
    return SHARQ_ECUDA;
  const int64_t m_pairs = (m_blocks + 1) / 2, n_tiles = (a.D + BN - 1) / BN;
  GemmParams pp{a.row_scale, a.w_ts, (const uint16_t*)a.bias, a.Y, a.ldy, (int32_t)a.T, (int32_t)a.D, (int32_t)a.K,
                a.out_dtype, (int32_t)m_blocks, (int32_t)(m_pairs * n_tiles), 0};
  const double a_pair = 256.0 * 1.5 * (double)a.K * 2.0;         // bf16 bytes of one 256-row block of both operands
  if (a_pair * (double)m_pairs > 48e6) {
    int64_t gm = (int64_t)(64e6 / a_pair);
    pp.group_m = (int32_t)(gm < 1 ? 1 : gm > m_pairs ? m_pairs : gm);
  }
  auto kfn = hif4_gemm_sp_pair_kernel<BN>;
  if (cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM) != cudaSuccess) return SHARQ_ECUDA;
  const int64_t tiles = m_pairs * n_tiles;
  const int64_t clusters = tiles < num_sms / 2 ? tiles : num_sms / 2;
  cudaLaunchConfig_t lp{};
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  lp.blockDim = dim3(kGemmThreads);
  lp.gridDim = dim3((unsigned)(2 * clusters));
  lp.dynamicSmemBytes = S::SMEM;
  lp.stream = st;
  lp.attrs = at;
  lp.numAttrs = 1;
  return cudaLaunchKernelEx(&lp, kfn, tm_asp, tm_adn, tm_w, tm_e, pp, (int)a.path) == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}
}  // namespace

sharq_status launch_linear_hif4(const LinearArgs& a, void* workspace, size_t workspace_bytes, int num_sms,
                                cudaStream_t st) {
  if (!workspace || workspace_bytes < hif4_linear_workspace_bytes(a.T, a.D, a.K)) return SHARQ_EWORKSPACE;
  if (a.K > (int64_t)1 << 24 || a.D > (int64_t)1 << 24 || a.T > (int64_t)1 << 30) return SHARQ_ESHAPE;
  const int64_t Tp = round_up(a.T, 128);
  uint16_t* A = reinterpret_cast<uint16_t*>((reinterpret_cast<uintptr_t>(workspace) + 127) & ~(uintptr_t)127);
  const uint16_t* W = reinterpret_cast<const uint16_t*>(a.w_sf_dn);   // bf16 [D, K], written by sharq_quantize_weight
  const int64_t na = a.T * (a.K >> 3);
  {
    const int64_t mb = Tp / 128;
    if (mb >= 2 && ((mb + 1) / 2) * ((a.D + 223) / 224) >= num_sms / 4 && a.K % 128 == 0)
      return a.D % 192 == 0 && a.D % 224 != 0 ? launch_sp_pair<192>(a, workspace, Tp, mb, num_sms, st)
                                              : launch_sp_pair<224>(a, workspace, Tp, mb, num_sms, st);
  }
  hif4_dequant_act_kernel<<<(unsigned)((na + 255) / 256 < 8192 ? (na + 255) / 256 : 8192), 256, 0, st>>>(
      (const uint8_t*)a.sp_codes, (const uint32_t*)a.sp_sf, (const uint8_t*)a.sp_meta, (const uint8_t*)a.dn_codes,
      (const uint32_t*)a.dn_sf, A, a.T, a.K, a.path);
  if (cudaGetLastError() != cudaSuccess) return SHARQ_ECUDA;
  CUtensorMap tm_a, tm_w;
  const bool wide = a.D % 256 == 0;
  if (!make_bf16_map(&tm_a, A, (uint64_t)Tp, (uint64_t)(2 * a.K), GM) ||
      !make_bf16_map(&tm_w, W, (uint64_t)a.D, (uint64_t)a.K, wide ? 256 : 128))
    return SHARQ_ECUDA;
  const int64_t m_blocks = Tp / 128;
  GemmParams p{a.row_scale, a.w_ts, (const uint16_t*)a.bias, a.Y, a.ldy, (int32_t)a.T, (int32_t)a.D, (int32_t)a.K,
               a.out_dtype, (int32_t)m_blocks, (int32_t)(m_blocks * (a.D / (wide ? 256 : 128))), 0};
  return wide ? launch_gemm<256>(tm_a, tm_w, p, num_sms, st) : launch_gemm<128>(tm_a, tm_w, p, num_sms, st);
}

// ---- sharq_linear_hif4_static: the same path with its scratch in a file-scope device array (no allocation) ---------
// For callers that cannot provide (or allocate) a workspace: code under CUDA-graph capture, tight serving loops,
// harnesses that forbid cudaMalloc.  The bf16 copy of the activation operands [roundup(T, 128), 2K] goes to
// g_hif4_scratch instead of a caller's workspace.  Every GPU that loads the library holds the array until exit.
// In HOST code the array's name is only a stand-in for the symbol, not a device address: the address is taken once per
// device, with that device current, by cudaGetSymbolAddress, and that pointer is what the kernels get.
constexpr size_t kHif4StaticScratchBytes = SHARQ_STATIC_SCRATCH_BYTES;
static __device__ __align__(256) uint8_t g_hif4_scratch[kHif4StaticScratchBytes];

namespace {
constexpr int kScratchDevices = 64;
std::atomic<void*> g_scratch_ptr[kScratchDevices];      // per device ordinal; filled idempotently, lock-free

sharq_status static_scratch_ptr(int dev, void** out) {
  void* ptr = (dev >= 0 && dev < kScratchDevices) ? g_scratch_ptr[dev].load(std::memory_order_acquire) : nullptr;
  if (!ptr) {
    if (cudaGetSymbolAddress(&ptr, g_hif4_scratch) != cudaSuccess || !ptr) return SHARQ_ECUDA;   // current device = dev
    if (dev >= 0 && dev < kScratchDevices) g_scratch_ptr[dev].store(ptr, std::memory_order_release);
  }
  *out = ptr;
  return SHARQ_OK;
}
}  // namespace

}  // namespace sharq

extern "C" sharq_status sharq_linear_hif4_static(const sharq_config* cfg, int64_t T, int64_t D, int64_t K,
                                                 const void* sp_codes, const void* sp_sf, const void* sp_meta,
                                                 const void* dn_codes, const void* dn_sf, const float* row_scale,
                                                 const void* w_codes, const void* w_sf_sparse_view,
                                                 const void* w_sf_dense_view, const float* w_tensor_scale,
                                                 const void* bias, void* Y, int64_t ldy, int32_t out_dtype,
                                                 int32_t path, void* stream) {
  using namespace sharq;
  if (!cfg || cfg->fmt != SHARQ_HIF4 || cfg->mask != SHARQ_MASK_24 || cfg->layout != SHARQ_LAYOUT_CANONICAL)
    return SHARQ_EINVAL;
  if (T < 0 || T >= (int64_t)1 << 30 || D <= 0 || D % 128 != 0 || K <= 0 || K % 256 != 0 || ldy < D || ldy % 8 != 0)
    return SHARQ_ESHAPE;
  if (out_dtype < 0 || out_dtype > 1 || path < 0 || path > 2) return SHARQ_EINVAL;
  if (T == 0) return SHARQ_OK;
  // the scratch is a fixed array: larger problems are refused, never silently truncated
  if (hif4_linear_workspace_bytes(T, D, K) > kHif4StaticScratchBytes) return SHARQ_EWORKSPACE;
  const void* ptrs[] = {sp_codes, sp_sf, sp_meta, dn_codes, dn_sf, w_codes, w_sf_sparse_view, w_sf_dense_view, Y};
  for (const void* q : ptrs)
    if (!q || (reinterpret_cast<uintptr_t>(q) & 15u)) return SHARQ_EINVAL;
  if (!row_scale || !w_tensor_scale) return SHARQ_EINVAL;
  int dev = 0, major = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return SHARQ_ECUDA;
  if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return SHARQ_ECUDA;
  if (major != 10) return SHARQ_EARCH;
  void* scratch = nullptr;
  const sharq_status s = static_scratch_ptr(dev, &scratch);
  if (s != SHARQ_OK) return s;
  // nothing in the scratch has to start at zero: rows 0 .. T-1 of the bf16 operand copy are rewritten by every call
  // before the GEMM reads them; the pad rows up to roundup(T, 128) keep an earlier call's bytes and only feed
  // accumulator rows that are never stored
  LinearArgs a{T, D, K, sp_codes, sp_sf, sp_meta, dn_codes, dn_sf, nullptr, row_scale, w_codes, w_sf_sparse_view,
               w_sf_dense_view, w_tensor_scale, bias, Y, ldy, out_dtype, path};
  return launch_linear_hif4(a, scratch, kHif4StaticScratchBytes, sms, (cudaStream_t)stream);
}
