// sharq_linear for decode shapes (T <= 64, NVFP4): operands swapped so that the MMA cost follows T.
//
// tcgen05.mma always spends max(M,128) * N / 256 cycles per K-chunk.  With the activations on the M side
// (as the sparse instruction demands: the 2:4-compressed operand must be A) a T = 1 layer pays for 128
// rows and the kernel is bound by MMA issue, not by the weight stream (measured: 0.43 us per 256-k block
// of a 128-wide tile against 0.12 us of HBM time).  Here the WEIGHT tile is A (M = 128 output features)
// and the activations are B (N = roundup(T, 8) columns): the same products cost N/128 of the cycles.  The
// price: the backbone can no longer use tcgen05.mma.sp, so the epilogue warps, idle during the main loop,
// expand the compressed backbone (codes + metadata) of each k-block into a dense FP4 operand in shared
// memory (zeros at the dropped pairs; at most 64 rows, a few KB) and duplicate its group-32 scales into
// the group-16 form the dense block-scaled MMA takes.  Mathematically identical to the sparse form
// (Eq. 9): every product is the same, only the fp32 summation order differs.
//
// Accumulator in TMEM: lane = output feature (W row), column = token.  Split-K over a cluster with a
// DSMEM exchange of 8-token slices as in linear.cu.  Warps: 0 = TMA producer, 1 = MMA issuer,
// 2-5 = backbone expanders during the main loop, then epilogue.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdlib.h>

#include "common.cuh"
#include "tc_ptx.cuh"

namespace sharq {

struct LinearArgs {
  int64_t T, D, K;
  const void *sp_codes, *sp_sf, *sp_meta, *dn_codes, *dn_sf;
  const float* row_scale;
  const void *w_codes, *w_sf_sp, *w_sf_dn;
  const float* w_ts;
  const void* bias;
  void* Y; int64_t ldy; int out_dtype; int path;
};

namespace {

constexpr int kThreads = 192;
constexpr int kTmemCols = 256;
constexpr int DK = 256;                 // logical k per ring stage

struct DParams {
  const uint8_t *sp_sf, *sp_meta, *dn_sf, *w_sf_dn;
  const float *row_scale, *w_ts;
  const uint16_t* bias;
  void* Y;
  int64_t ldy;
  int32_t T, D, K, out_fp32, path, n_cols, tiles;     // n_cols = roundup(T, 8): the MMA's N
  int32_t no_mma;     // experiment: consume the ring without issuing any tensor-core work
  int32_t w_tiled;    // weight codes stored as [D/128][K/256] tiles of 128 rows x 128 B (16 KB contiguous)
};

template <int NMAX, bool SPLIT>
struct DStage {
  static constexpr int W = 0;                          // 128 weight rows x 128 B, SW128   (A operand)
  static constexpr int B_DN = W + 128 * 128;           // residual codes, n_cols rows x 128 B, SW128
  static constexpr int B_SP = B_DN + NMAX * 128;       // expanded backbone, same layout (written by warps 2-5)
  static constexpr int SFA = B_SP + NMAX * 128;        // W dense-view scales: 4 atoms
  static constexpr int SFB_DN = SFA + 2048;            // residual scales: 4 atoms
  static constexpr int SFB_SP = SFB_DN + 2048;         // backbone scales duplicated to group 16: 4 atoms
  static constexpr int RAW_C = SFB_SP + 2048;          // compressed backbone codes, n_cols rows x 64 B, linear
  static constexpr int RAW_META = RAW_C + NMAX * 64;   // metadata tile (128 rows x 16 B)
  static constexpr int RAW_SF = RAW_META + 2048;       // backbone scales: 2 atoms
  static constexpr int RAW = RAW_SF + 1024;
  static constexpr int BYTES = (RAW + 1023) / 1024 * 1024;
  static constexpr int RECV = SPLIT ? 9 * 128 * 32 : 0;            // [src][slot][128 lanes][8 fp32]
  static constexpr int PAD = 8 * 1024;                             // B tiles are read as >= 8 rows
  static constexpr int FIT = (232448 - 1024 - 256 - RECV - PAD) / BYTES;
  static constexpr int STAGES = FIT > 8 ? 8 : FIT;
  static constexpr int SMEM = STAGES * BYTES + PAD + RECV + 1024 + 256;
  static constexpr int ACC_STRIDE = 64;                // two accumulator stages of <= 64 columns
  static constexpr int SFA_COL = 128, SFB_DN_COL = 144, SFB_SP_COL = 160;
};

template <int NMAX, bool SPLIT>
__global__ void __launch_bounds__(kThreads, 1)
sharq_linear_decode_kernel(const __grid_constant__ CUtensorMap tm_w, const __grid_constant__ CUtensorMap tm_dn,
                           const __grid_constant__ CUtensorMap tm_spc, const DParams p) {
  using S = DStage<NMAX, SPLIT>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* const smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));      // generic pointer to the same place
  const uint32_t recv_base = smem_base + S::STAGES * S::BYTES + S::PAD;
  const uint32_t bars = recv_base + S::RECV;
  auto full_bar = [&](int s) { return bars + 8u * s; };
  auto exp_bar = [&](int s) { return bars + 8u * (S::STAGES + s); };
  auto empty_bar = [&](int s) { return bars + 8u * (2 * S::STAGES + s); };
  auto tmem_full_bar = [&](int a) { return bars + 8u * (3 * S::STAGES + a); };
  auto tmem_empty_bar = [&](int a) { return bars + 8u * (3 * S::STAGES + 2 + a); };
  const uint32_t tmem_ptr_smem = bars + 8u * (3 * S::STAGES + 4);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const bool do_sp = p.path != 2, do_dn = p.path != 1;
  const int N = p.n_cols;
  const int num_kb = p.K / DK;
  const int rank = SPLIT ? (int)tc::cluster_ctarank() : 0;
  const int splits = SPLIT ? (int)tc::cluster_nctarank() : 1;
  const int tile0 = SPLIT ? (int)tc::cluster_id_x() : (int)blockIdx.x;
  const int tile_step = SPLIT ? p.tiles : (int)gridDim.x;
  const int kb0 = (int)((int64_t)rank * num_kb / splits), kb1 = (int)((int64_t)(rank + 1) * num_kb / splits);

  if (warp == 0 && lane == 0) {
    tc::prefetch_tmap(&tm_w);
    tc::prefetch_tmap(&tm_dn);
    tc::prefetch_tmap(&tm_spc);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < S::STAGES; ++s) {
      tc::mbar_init(full_bar(s), 1);
      tc::mbar_init(exp_bar(s), 4);             // one arrival per expander warp
      tc::mbar_init(empty_bar(s), 1);
    }
    for (int a = 0; a < 2; ++a) {
      tc::mbar_init(tmem_full_bar(a), 1);
      tc::mbar_init(tmem_empty_bar(a), 4);
    }
    tc::fence_mbar_init();
  }
  if (warp == 2) tc::tmem_alloc<kTmemCols>(tmem_ptr_smem);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_smem));
  tc::grid_launch_dependents();

  if (warp == 0) {
    // =========================== TMA producer ===============================================
    const bool lead = tc::elect_one() != 0;
    const uint64_t pol_w = tc::policy_evict_first(), pol_a = tc::policy_evict_last();
    const int64_t Kc = p.K;
    uint32_t tx = 128 * 128 + 2048;                                   // W tile + its dense-view scales
    if (do_dn) tx += N * 128 + 2048;
    if (do_sp) tx += N * 64 + 2048 + 1024;
    uint32_t it = 0;
    bool dep_synced = false;
    for (int tile = tile0; tile < p.tiles; tile += tile_step) {
      const int n0 = tile * 128;                                      // first output feature of the tile
      auto load_w = [&](int kb, uint32_t st, uint32_t fb) {
        if (lead) tc::tma_load_2d(st + S::W, &tm_w, fb, p.w_tiled ? 0 : kb * 128,
                                  p.w_tiled ? (tile * (p.K / 256) + kb) * 128 : n0, pol_w);
        if (lead) tc::bulk_load(st + S::SFA, p.w_sf_dn + ((size_t)tile * (Kc / 256) + (size_t)kb) * 2048, 2048, fb, pol_w);
      };
      auto load_a = [&](int kb, uint32_t st, uint32_t fb) {
        if (do_dn) {
          if (lead) tc::tma_load_2d(st + S::B_DN, &tm_dn, fb, kb * 128, 0, pol_a);
          if (lead) tc::bulk_load(st + S::SFB_DN, p.dn_sf + (size_t)kb * 2048, 2048, fb, pol_a);
        }
        if (do_sp) {
          if (lead) tc::tma_load_2d(st + S::RAW_C, &tm_spc, fb, kb * 64, 0, pol_a);
          if (lead) tc::bulk_load(st + S::RAW_META, p.sp_meta + (size_t)kb * 2048, 2048, fb, pol_a);
          if (lead) tc::bulk_load(st + S::RAW_SF, p.sp_sf + (size_t)kb * 1024, 1024, fb, pol_a);
        }
      };
      int kb = kb0;
      if (!dep_synced) {                       // PDL: weights first, activations after the producer kernel is done
        const int n_early = min(S::STAGES, kb1 - kb0);
        for (int i = 0; i < n_early; ++i) {
          if (lead) tc::mbar_expect_tx(full_bar(i), tx);
          load_w(kb + i, smem_base + i * S::BYTES, full_bar(i));
        }
        tc::grid_dependency_wait();
        dep_synced = true;
        for (int i = 0; i < n_early; ++i) load_a(kb + i, smem_base + i * S::BYTES, full_bar(i));
        kb += n_early;
        it += n_early;
      }
      for (; kb < kb1; ++kb, ++it) {
        const int s = it % S::STAGES;
        tc::mbar_wait(empty_bar(s), ((it / S::STAGES) & 1) ^ 1);
        const uint32_t st = smem_base + s * S::BYTES;
        if (lead) tc::mbar_expect_tx(full_bar(s), tx);
        load_w(kb, st, full_bar(s));
        load_a(kb, st, full_bar(s));
      }
    }
    if (!dep_synced) tc::grid_dependency_wait();
  } else if (warp == 1) {
    // =========================== MMA issuer =================================================
    const bool lead = tc::elect_one() != 0;
    const uint32_t idesc = tc::idesc_fp4(128, (uint32_t)N, false, false, 0, 0);
    uint32_t it = 0, n_unit = 0;
    for (int tile = tile0; tile < p.tiles; tile += tile_step, ++n_unit) {
      const uint32_t as = n_unit & 1u;
      const uint32_t acc = tmem_base + as * S::ACC_STRIDE;
      tc::mbar_wait(tmem_empty_bar(as), ((n_unit >> 1) & 1u) ^ 1u);
      tc::tc_fence_after();
      uint32_t accumulate = 0;
      for (int kb = kb0; kb < kb1; ++kb, ++it) {
        const int s = it % S::STAGES;
        const uint32_t ph = (it / S::STAGES) & 1;
        tc::mbar_wait(full_bar(s), ph);
        if (do_sp) tc::mbar_wait(exp_bar(s), ph);
        tc::tc_fence_after();
        const uint32_t st = smem_base + s * S::BYTES;
        if (p.no_mma) {
          if (lead) tc::mbar_arrive(empty_bar(s));
          continue;
        }
#pragma unroll
        for (int a = 0; a < 4; ++a) {
          if (lead) tc::tc_cp_sf(tmem_base + S::SFA_COL + 4 * a, tc::smem_desc(st + S::SFA + 512 * a, 128, 0));
          if (do_dn && lead) tc::tc_cp_sf(tmem_base + S::SFB_DN_COL + 4 * a, tc::smem_desc(st + S::SFB_DN + 512 * a, 128, 0));
          if (do_sp && lead) tc::tc_cp_sf(tmem_base + S::SFB_SP_COL + 4 * a, tc::smem_desc(st + S::SFB_SP + 512 * a, 128, 0));
        }
        if (do_dn) {
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            if (lead) tc::mma_dense<true>(acc, tc::smem_desc(st + S::W + 32 * j, 1024, 2),
                                          tc::smem_desc(st + S::B_DN + 32 * j, 1024, 2), idesc,
                                          tmem_base + S::SFA_COL + 4 * j, tmem_base + S::SFB_DN_COL + 4 * j, accumulate);
            accumulate = 1;
          }
        }
        if (do_sp) {
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            if (lead) tc::mma_dense<true>(acc, tc::smem_desc(st + S::W + 32 * j, 1024, 2),
                                          tc::smem_desc(st + S::B_SP + 32 * j, 1024, 2), idesc,
                                          tmem_base + S::SFA_COL + 4 * j, tmem_base + S::SFB_SP_COL + 4 * j, accumulate);
            accumulate = 1;
          }
        }
        if (lead) tc::tc_commit(empty_bar(s));
      }
      if (lead) tc::tc_commit(tmem_full_bar(as));
    }
  } else {
    // ============ backbone expanders during the main loop, then epilogue ======================
    const int tid = (int)threadIdx.x - 64;               // 0..127
    const int sub = warp & 3, n_local = sub * 32 + lane; // TMEM lane = output feature inside the tile
    const uint32_t lane_addr = tmem_base + ((uint32_t)(sub * 32) << 16);
    tc::grid_dependency_wait();                          // row_scale / Y belong to the kernels before us
    const float w_ts = p.w_ts[0];
    uint32_t it = 0, n_unit = 0;
    for (int tile = tile0; tile < p.tiles; tile += tile_step, ++n_unit) {
      if (do_sp) {
        for (int kb = kb0; kb < kb1; ++kb, ++it) {
          const int s = it % S::STAGES;
          tc::mbar_wait(full_bar(s), (it / S::STAGES) & 1);
          uint8_t* st = smem_gen + (size_t)s * S::BYTES;
          for (int item = tid; item < N * 8; item += 128) {
            const int r = item >> 3, u = item & 7;       // row, 16-byte unit (32 logical k = 4 chunks)
            const uint2 comp = *reinterpret_cast<const uint2*>(st + S::RAW_C + r * 64 + u * 8);
            const uint32_t meta = *reinterpret_cast<const uint16_t*>(st + S::RAW_META + r * 16 + u * 2);
            uint32_t w[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              const uint32_t nib = (meta >> (4 * c)) & 15u, i0 = nib & 3u, i1 = nib >> 2;
              const uint32_t two = ((c < 2 ? comp.x : comp.y) >> (16 * (c & 1))) & 0xFFFFu;
              w[c] = ((two & 0xFFu) << (8 * i0)) | ((two >> 8) << (8 * i1));   // kept pairs in place, zeros elsewhere
            }
            *reinterpret_cast<uint4*>(st + S::B_SP + r * 128 + ((u ^ (r & 7)) << 4)) = make_uint4(w[0], w[1], w[2], w[3]);
          }
          if (tid < N) {                                 // group-32 scales -> group-16 (each used twice)
            const int off = (tid & 31) * 16 + (tid >> 5) * 4;
            const uint32_t in0 = *reinterpret_cast<const uint32_t*>(st + S::RAW_SF + off);
            const uint32_t in1 = *reinterpret_cast<const uint32_t*>(st + S::RAW_SF + 512 + off);
            *reinterpret_cast<uint32_t*>(st + S::SFB_SP + off) = __byte_perm(in0, 0u, 0x1100u);
            *reinterpret_cast<uint32_t*>(st + S::SFB_SP + 512 + off) = __byte_perm(in0, 0u, 0x3322u);
            *reinterpret_cast<uint32_t*>(st + S::SFB_SP + 1024 + off) = __byte_perm(in1, 0u, 0x1100u);
            *reinterpret_cast<uint32_t*>(st + S::SFB_SP + 1536 + off) = __byte_perm(in1, 0u, 0x3322u);
          }
          tc::fence_proxy_async();                       // generic-proxy writes -> visible to tcgen05
          __syncwarp();
          if (lane == 0) tc::mbar_arrive(exp_bar(s));
        }
      }
      const uint32_t as = n_unit & 1u;
      const int n_glob = tile * 128 + n_local;
      tc::mbar_wait(tmem_full_bar(as), (n_unit >> 1) & 1u);
      tc::tc_fence_after();
      const int slots = SPLIT ? (N / 8 + splits - 1) / splits : 0;
      for (int j = 0; j < N / 8; ++j) {
        uint32_t v[8];
        tc::tmem_ld8(lane_addr + as * S::ACC_STRIDE + j * 8, v);
        tc::tmem_ld_wait();
        if constexpr (SPLIT) {
          const uint32_t local = recv_base + (uint32_t)(((rank * slots + j / splits) * 128 + n_local) * 32);
          const uint32_t remote = tc::map_to_cta(local, (uint32_t)(j % splits));
          tc::st_cluster_v4(remote, __uint_as_float(v[0]), __uint_as_float(v[1]), __uint_as_float(v[2]), __uint_as_float(v[3]));
          tc::st_cluster_v4(remote + 16, __uint_as_float(v[4]), __uint_as_float(v[5]), __uint_as_float(v[6]), __uint_as_float(v[7]));
        } else {
          const float bias = p.bias ? __uint_as_float((uint32_t)p.bias[n_glob] << 16) : 0.0f;
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int t = j * 8 + i;
            if (t < p.T) {
              float y = __fmul_rn(__uint_as_float(v[i]), __fmul_rn(p.row_scale[t], w_ts));
              if (p.bias) y = __fadd_rn(y, bias);
              if (p.out_fp32) static_cast<float*>(p.Y)[(int64_t)t * p.ldy + n_glob] = y;
              else static_cast<uint16_t*>(p.Y)[(int64_t)t * p.ldy + n_glob] = (uint16_t)(pack_bf16x2_rn(y, 0.0f) & 0xFFFFu);
            }
          }
        }
      }
      tc::tc_fence_before();
      __syncwarp();
      if (lane == 0) tc::mbar_arrive(tmem_empty_bar(as));
    }
  }
  if constexpr (SPLIT) {
    __syncwarp();
    tc::cluster_sync_all();                              // partial slices have landed in their owners
    if (warp >= 2) {
      const int n_local = (warp & 3) * 32 + lane, n_glob = tile0 * 128 + n_local;
      const int slots = (N / 8 + splits - 1) / splits;
      const float w_ts = p.w_ts[0];
      const float bias = p.bias ? __uint_as_float((uint32_t)p.bias[n_glob] << 16) : 0.0f;
      for (int slot = 0; slot < slots; ++slot) {
        const int j = slot * splits + rank;              // the 8-token slices this CTA owns
        if (j >= N / 8) break;
        float f[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) f[i] = 0.0f;
        for (int src = 0; src < splits; ++src) {         // fixed order: deterministic sum
          const uint32_t a = recv_base + (uint32_t)(((src * slots + slot) * 128 + n_local) * 32);
          const float4 lo = tc::ld_shared_v4(a), hi = tc::ld_shared_v4(a + 16);
          f[0] = __fadd_rn(f[0], lo.x); f[1] = __fadd_rn(f[1], lo.y); f[2] = __fadd_rn(f[2], lo.z); f[3] = __fadd_rn(f[3], lo.w);
          f[4] = __fadd_rn(f[4], hi.x); f[5] = __fadd_rn(f[5], hi.y); f[6] = __fadd_rn(f[6], hi.z); f[7] = __fadd_rn(f[7], hi.w);
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const int t = j * 8 + i;
          if (t < p.T) {
            float y = __fmul_rn(f[i], __fmul_rn(p.row_scale[t], w_ts));
            if (p.bias) y = __fadd_rn(y, bias);
            if (p.out_fp32) static_cast<float*>(p.Y)[(int64_t)t * p.ldy + n_glob] = y;
            else static_cast<uint16_t*>(p.Y)[(int64_t)t * p.ldy + n_glob] = (uint16_t)(pack_bf16x2_rn(y, 0.0f) & 0xFFFFu);
          }
        }
      }
    }
  }
  __syncthreads();
  if (warp == 2) {
    tc::tc_fence_after();
    tc::tmem_dealloc<kTmemCols>(tmem_base);
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

bool make_byte_map(CUtensorMap* m, const void* base, uint64_t rows, uint64_t row_bytes, uint32_t box_bytes,
                   uint32_t box_rows, CUtensorMapSwizzle sw) {
  static EncodeTiledFn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      f = nullptr;
    return reinterpret_cast<EncodeTiledFn>(f);
  }();
  if (!fn) return false;
  cuuint64_t dims[2] = {row_bytes, rows};
  cuuint64_t strides[1] = {row_bytes};
  cuuint32_t box[2] = {box_bytes, box_rows};
  cuuint32_t estr[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// largest cluster size in {8, 4, 3, 2} for which all `tiles` clusters are co-resident in one wave
template <int NMAX>
int decode_splits(int64_t tiles, int num_kb, int num_sms) {
  if (tiles * 2 > num_sms) return 1;
  using S = DStage<NMAX, true>;
  static int max_clusters[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
  const int cand[4] = {8, 4, 3, 2};
  for (int c : cand) {
    if (tiles * c > num_sms || num_kb < 2 * c) continue;
    if (max_clusters[c] == 0) {
      cudaLaunchConfig_t lc{};
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = (unsigned)c; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      lc.gridDim = dim3((unsigned)(c * num_sms)); lc.blockDim = dim3(kThreads); lc.dynamicSmemBytes = S::SMEM;
      lc.attrs = at; lc.numAttrs = 1;
      int n = 0;
      auto kfn = sharq_linear_decode_kernel<NMAX, true>;
      cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM);
      if (cudaOccupancyMaxActiveClusters(&n, kfn, &lc) != cudaSuccess || n <= 0) n = -1;
      max_clusters[c] = n;
    }
    if (max_clusters[c] >= tiles) return c;
  }
  return 1;
}

template <int NMAX>
sharq_status launch_decode(const LinearArgs& a, const DParams& p, const CUtensorMap& tm_w, const CUtensorMap& tm_dn,
                           const CUtensorMap& tm_spc, int num_sms, cudaStream_t st) {
  const int splits = decode_splits<NMAX>(p.tiles, (int)(a.K / DK), num_sms);
  cudaLaunchConfig_t lc{};
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = attr;
  lc.numAttrs = 1;
  lc.blockDim = dim3(kThreads);
  lc.stream = st;
  if (splits > 1) {
    using S = DStage<NMAX, true>;
    auto kfn = sharq_linear_decode_kernel<NMAX, true>;
    if (cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM) != cudaSuccess)
      return SHARQ_ECUDA;
    lc.gridDim = dim3((unsigned)(p.tiles * splits));
    lc.dynamicSmemBytes = S::SMEM;
    attr[1].id = cudaLaunchAttributeClusterDimension;
    attr[1].val.clusterDim.x = (unsigned)splits;
    attr[1].val.clusterDim.y = 1;
    attr[1].val.clusterDim.z = 1;
    lc.numAttrs = 2;
    return cudaLaunchKernelEx(&lc, kfn, tm_w, tm_dn, tm_spc, p) == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
  }
  using S = DStage<NMAX, false>;
  auto kfn = sharq_linear_decode_kernel<NMAX, false>;
  if (cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM) != cudaSuccess)
    return SHARQ_ECUDA;
  lc.gridDim = dim3((unsigned)(p.tiles < num_sms ? p.tiles : num_sms));
  lc.dynamicSmemBytes = S::SMEM;
  return cudaLaunchKernelEx(&lc, kfn, tm_w, tm_dn, tm_spc, p) == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}

}  // namespace

// NVFP4, one problem (no experts), T <= 64.  Called by launch_linear (linear.cu).
sharq_status launch_linear_decode(const LinearArgs& a, int num_sms, cudaStream_t st) {
  const int n_cols = (int)((a.T + 7) / 8 * 8);
  CUtensorMap tm_w, tm_dn, tm_spc;
  const bool w_tiled = getenv("SHARQ_EXP_WTILED") != nullptr;
  if (!(w_tiled ? make_byte_map(&tm_w, a.w_codes, (uint64_t)a.D * (uint64_t)(a.K / 256), 128, 128, 128, CU_TENSOR_MAP_SWIZZLE_128B)
                : make_byte_map(&tm_w, a.w_codes, (uint64_t)a.D, (uint64_t)a.K / 2, 128, 128, CU_TENSOR_MAP_SWIZZLE_128B)) ||
      !make_byte_map(&tm_dn, a.dn_codes, (uint64_t)a.T, (uint64_t)a.K / 2, 128, (uint32_t)n_cols,
                     CU_TENSOR_MAP_SWIZZLE_128B) ||
      !make_byte_map(&tm_spc, a.sp_codes, (uint64_t)a.T, (uint64_t)a.K / 4, 64, (uint32_t)n_cols,
                     CU_TENSOR_MAP_SWIZZLE_NONE))
    return SHARQ_ECUDA;
  DParams p{(const uint8_t*)a.sp_sf, (const uint8_t*)a.sp_meta, (const uint8_t*)a.dn_sf, (const uint8_t*)a.w_sf_dn,
            a.row_scale, a.w_ts, (const uint16_t*)a.bias, a.Y, a.ldy, (int32_t)a.T, (int32_t)a.D, (int32_t)a.K,
            a.out_dtype, a.path, n_cols, (int32_t)(a.D / 128), getenv("SHARQ_EXP_NOMMA") ? 1 : 0, w_tiled ? 1 : 0};
  return n_cols <= 16 ? launch_decode<16>(a, p, tm_w, tm_dn, tm_spc, num_sms, st)
                      : launch_decode<64>(a, p, tm_w, tm_dn, tm_spc, num_sms, st);
}

}  // namespace sharq
