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
#include "prepare_device.cuh"

namespace sharq {

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
        if (p.combo) quantize_block_combo<FMT>(p, row, (uint32_t)k0, X, ts, inv_ts);
        else if (p.mask24) quantize_block_e2m1_24<FMT>(p, row, (uint32_t)k0, X, ts, inv_ts);
        else quantize_block_e2m1<FMT>(p, row, (uint32_t)k0, X, ts, inv_ts);
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

// ---- row-per-CTA kernel (K <= 32768): body in prepare_device.cuh --------------------------------------
template <int FMT, int NORM, int MAXT, int MINB, bool SWIGLU = false>
__global__ void __launch_bounds__(MAXT, MINB) sharq_prepare_row_kernel(const PrepParams p) {
  extern __shared__ __align__(16) uint8_t row_smem[];
  // programmatic dependent launch: let the GEMM that follows start streaming its weights now; our own
  // inputs (and the operand buffers we overwrite) belong to the kernels before us
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  prepare_rows<FMT, NORM, 0, (MAXT >= 512), SWIGLU>(p, row_smem, (int)threadIdx.x, (int)blockDim.x, (int64_t)blockIdx.x, (int64_t)gridDim.x);
}

template <int FMT>
static cudaError_t launch_row_kernel(int norm, const PrepParams& p, int num_sms, cudaStream_t st);

// dynamic shared memory of the row-per-CTA kernel for rows of `warps` 1024-element blocks (prepare_rows' layout)
static size_t row_kernel_smem(int fmt, int norm, int warps) {
  return (size_t)warps * 1024 + 256 + 16 + 64                                                         // leaves, amax, stat, mask table
         + (size_t)warps * 32 * (norm == SHARQ_NORM_LAYER ? 128 : norm == SHARQ_NORM_RMS ? 64 : 0)    // gamma, beta
         + (fmt == SHARQ_NVFP4 && warps > 8 ? (size_t)warps * 32 * 128 + 512 + 16 : 0);   // lagged loop: parked row (2 stages), amax slots, mbarriers
}
constexpr size_t kRowKernelSmemMax = 227 * 1024;   // opt-in limit per CTA on sm_100

// The row kernel indexes with 32 bits: at most 2^31 / max(ldx, K) rows (a multiple of 128, so the tiled
// layouts split at tile boundaries) per launch; larger problems run as several launches on row ranges.
template <int FMT>
static cudaError_t launch_row_chunks(int norm, const PrepParams& p0, int num_sms, cudaStream_t st) {
  int64_t widest = p0.ldx > p0.K ? p0.ldx : p0.K;
  if (p0.res) { if (p0.ldr > widest) widest = p0.ldr; if (p0.ldo > widest) widest = p0.ldo; }
  int64_t max_rows = ((int64_t(1) << 31) / widest) & ~int64_t(127);
  if (debug_env().prep_chunk_rows > 0) max_rows = (int64_t)debug_env().prep_chunk_rows & ~int64_t(127);
  if (max_rows < 128) return cudaErrorInvalidValue;
  const int64_t K = p0.K;
  for (int64_t r0 = 0; r0 < p0.T; r0 += max_rows) {
    PrepParams p = p0;
    p.T = (p0.T - r0 < max_rows) ? p0.T - r0 : max_rows;
    p.x = p0.x + r0 * p0.ldx;
    if (p0.res) { p.res = p0.res + r0 * p0.ldr; p.sum_out = p0.sum_out + r0 * p0.ldo; }
    p.sp_codes = p0.sp_codes + r0 * (K >> 2);
    p.dn_codes = p0.dn_codes + r0 * (K >> 1);
    p.row_scale = p0.row_scale + r0;
    if (FMT == SHARQ_HIF4) {                       // canonical only: metadata K/8 bytes, scale words K/64 per row
      p.sp_meta = p0.sp_meta + r0 * (K >> 3);
      p.sp_sf = p0.sp_sf + r0 * (K >> 6) * 4;
      p.dn_sf = p0.dn_sf + r0 * (K >> 6) * 4;
    } else {                                       // r0 % 128 == 0: both layouts advance by whole rows / tiles
      const int64_t c_dn = (FMT == SHARQ_NVFP4) ? (K >> 4) : (K >> 5);
      p.sp_meta = p0.sp_meta + r0 * (K >> 4);
      p.sp_sf = p0.sp_sf + r0 * (K >> 5);
      p.dn_sf = p0.dn_sf + r0 * c_dn;
    }
    const cudaError_t e = launch_row_kernel<FMT>(norm, p, num_sms, st);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
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
  lc.dynamicSmemBytes = row_kernel_smem(FMT, norm, warps);
  cudaError_t err = cudaSuccess;
  const bool swiglu = p.res != nullptr && p.sum_out == nullptr;        // sharq_prepare_swiglu (norm NONE only, checked by the C ABI)
#define SHARQ_ROW(N, MAXT, MINB)                                                                              \
  do {                                                                                                        \
    auto kfn = sharq_prepare_row_kernel<FMT, N, MAXT, MINB>;                                                  \
    if (lc.dynamicSmemBytes > 48 * 1024)                                                                      \
      err = cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)lc.dynamicSmemBytes); \
    if (err == cudaSuccess) err = cudaLaunchKernelEx(&lc, kfn, p);                                            \
  } while (0)
#define SHARQ_ROW_SWIGLU(MAXT, MINB)                                                                         \
  do {                                                                                                        \
    auto kfn = sharq_prepare_row_kernel<FMT, SHARQ_NORM_NONE, MAXT, MINB, true>;                              \
    if (lc.dynamicSmemBytes > 48 * 1024)                                                                      \
      err = cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)lc.dynamicSmemBytes); \
    if (err == cudaSuccess) err = cudaLaunchKernelEx(&lc, kfn, p);                                            \
  } while (0)
#define SHARQ_ROW_N(MAXT, MINB)                                              \
  {                                                                          \
    if (swiglu) SHARQ_ROW_SWIGLU(MAXT, MINB);                                \
    else if (norm == SHARQ_NORM_NONE) SHARQ_ROW(SHARQ_NORM_NONE, MAXT, MINB); \
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
#undef SHARQ_ROW_SWIGLU
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

// Kernel parameters of a plain sharq_prepare (also used by sharq_prepare_linear's in-kernel rows, linear.cu)
PrepParams make_prep_params(const sharq_config* cfg, const void* x, int64_t T, int64_t K, int64_t ldx, const void* gamma,
                            const void* beta, const float* x_ts, void* sp_codes, void* sp_sf, void* sp_meta,
                            void* dn_codes, void* dn_sf, float* row_scale) {
  PrepParams p;
  p.res = nullptr; p.sum_out = nullptr; p.ldr = 0; p.ldo = 0;
  p.x = (const uint16_t*)x; p.ldx = ldx; p.T = T; p.K = K;
  p.gamma = (const uint16_t*)gamma; p.beta = (const uint16_t*)beta; p.x_ts = x_ts;
  p.sp_codes = (uint8_t*)sp_codes; p.sp_sf = (uint8_t*)sp_sf; p.sp_meta = (uint8_t*)sp_meta;
  p.dn_codes = (uint8_t*)dn_codes; p.dn_sf = (uint8_t*)dn_sf; p.row_scale = row_scale;
  p.eps = cfg->eps; p.tiled = (cfg->layout == SHARQ_LAYOUT_TILED);
  p.row_bytes = (uint32_t)(K * 2);
  p.nbuf = 0;
  p.idx_tags = 0x0004080Cu;
  p.mask24 = (cfg->fmt != SHARQ_HIF4 && cfg->mask == SHARQ_MASK_24) ? 1 : 0;
  p.combo = 0; p.dn_meta = nullptr;
  return p;
}

// Host launcher, called by the C ABI in api.cu after argument validation.
cudaError_t launch_prepare(const sharq_config* cfg, const void* x, int64_t T, int64_t K, int64_t ldx,
                           const void* gamma, const void* beta, const float* x_ts, void* sp_codes, void* sp_sf,
                           void* sp_meta, void* dn_codes, void* dn_sf, float* row_scale, int num_sms,
                           cudaStream_t st, const void* residual, int64_t ldr, void* sum_out, int64_t ldo,
                           int combo, void* dn_meta) {
  PrepParams p = make_prep_params(cfg, x, T, K, ldx, gamma, beta, x_ts, sp_codes, sp_sf, sp_meta, dn_codes, dn_sf, row_scale);
  p.combo = combo; p.dn_meta = (uint8_t*)dn_meta;
  p.res = (const uint16_t*)residual; p.sum_out = (uint16_t*)sum_out; p.ldr = ldr; p.ldo = ldo;
  // the row kernel reads 32 bytes per load: rows must start on 32-byte boundaries, otherwise (16-byte aligned
  // input, the C ABI's minimum) the warp-per-row kernel with its 16-byte cp.async takes the call
  const bool wide_ok = ((uintptr_t)x % 32 == 0) && (ldx % 16 == 0);
  // NVFP4 + LayerNorm on the widest rows (K > 25600): gamma, beta and the lagged loop's parked row together exceed the
  // shared memory of one CTA; those shapes go to the warp-per-row kernel (the fused-operand calls refuse them)
  const bool row_fits = K <= 1024 * kRowMaxWarps &&
                        row_kernel_smem(cfg->fmt, cfg->norm, (int)((K + 1023) / 1024)) <= kRowKernelSmemMax;
  if (residual && (!wide_ok || !row_fits || p.mask24 || combo)) return cudaErrorInvalidValue;   // checked by the C ABI
  if (row_fits && wide_ok && !p.mask24 && !combo && (!debug_env().old_prepare || residual)) {
    p.nbuf = 0;
    if (cfg->fmt == SHARQ_NVFP4) return launch_row_chunks<SHARQ_NVFP4>(cfg->norm, p, num_sms, st);
    if (cfg->fmt == SHARQ_MXFP4) return launch_row_chunks<SHARQ_MXFP4>(cfg->norm, p, num_sms, st);
    return launch_row_chunks<SHARQ_HIF4>(cfg->norm, p, num_sms, st);
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
    hif4_quant32<false>(X, v16, hs, c, e8b, e16b, nullptr, nullptr, nullptr, nullptr);
    const uint32_t word = hif4_meta_word(hs.e6m2, e8b, e16b, lane);
    if (!act) return;
    *reinterpret_cast<uint4*>(codes + d * (K >> 1) + (k0 >> 1)) = make_uint4(c[0], c[1], c[2], c[3]);
    if ((lane & 1) == 0) reinterpret_cast<uint32_t*>(sf_sp)[d * (K >> 6) + (k0 >> 6)] = word;
    return;                                         // the dense view (exact bf16 values) is written by a second kernel
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

cudaError_t launch_hif4_dequant_weight(const void* codes, const void* sf, void* W_bf16, int64_t D, int64_t K, cudaStream_t st);

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
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  // HiF4: the GEMM-side ("dense") view of the payload is its exact bf16 dequantisation, made once here
  if (cfg->fmt == SHARQ_HIF4) return launch_hif4_dequant_weight(codes, sf_sp, sf_dn, D, K, st);
  return cudaSuccess;
}

// ---- test helpers: TILED -> canonical (include/sharq.h "Output layouts"); pure index maps --------------------------
__global__ void untile_kernel(const uint8_t* __restrict__ tiled, int64_t R, int64_t C, uint8_t* __restrict__ canonical,
                              int meta) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < R * C; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / C, c = i % C;
    canonical[i] = tiled[meta ? meta_tiled_offset(r, c, C * 16) : sf_tiled_offset(r, c, C)];
  }
}

cudaError_t launch_untile(const void* tiled, int64_t R, int64_t C, void* canonical, int meta, cudaStream_t st) {
  const int64_t n = R * C;
  const unsigned blocks = (unsigned)((n + 255) / 256 < 4096 ? (n + 255) / 256 : 4096);
  untile_kernel<<<blocks, 256, 0, st>>>((const uint8_t*)tiled, R, C, (uint8_t*)canonical, meta);
  return cudaGetLastError();
}

}  // namespace sharq
