// sharq_linear / sharq_linear_grouped (Eq. 9): the sparse backbone GEMM and the dense
// residual GEMM of one SharQ linear layer, fused in ONE kernel.
//
// Per 128 x BN output tile one CTA streams K in blocks of 256 logical elements through a TMA-fed
// shared-memory ring.  Each W tile is loaded ONCE per k-block and consumed by both paths (P:157
// "single shared FP4 weight payload"): two tcgen05.mma.sp (K = 128 logical each, compressed A +
// metadata in tensor memory, one scale per 32 logical k) and four dense block-scaled tcgen05.mma
// (K = 64 each, one scale per 16) accumulate into the SAME fp32 TMEM tile ("accumulates
// directly into this output").  Scale factors and metadata arrive in the tcgen05 atom layouts
// sharq_prepare / sharq_quantize_weight emit (LAYOUT_TILED) so they go HBM -> smem with 1-D bulk
// copies and smem -> TMEM with tcgen05.cp, no re-formatting.  Epilogue: TMEM -> registers,
// y = acc * (row_scale[t] * w_tensor_scale) (+ bias), bf16 or fp32 store.
//
// Warp roles (192 threads): warp 0 = TMA producer, warp 1 = MMA issuer (one elected lane),
// warps 2-5 = epilogue (warp w owns TMEM lanes 32*(w%4)..+31); warp 2 also owns the TMEM allocation.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdlib.h>

#include <atomic>

#include "common.cuh"
#include "debug_env.h"
#include "linear_args.h"
#include "prepare_device.cuh"
#include "tc_ptx.cuh"
#include "epilogue.cuh"

namespace sharq {

namespace {

constexpr int kMaxExperts = 1024;  // the expert table lives in shared memory (2 x (E + 1) words per CTA)
constexpr int BM = 128;          // rows of an output tile = TMEM lanes
constexpr int BK = 256;          // logical k per pipeline stage
constexpr int kThreads = 192;

#if defined(SHARQ_EXPERIMENTS) && defined(SHARQ_DEBUG_TS)   // experiments only: per-CTA phase timestamps (SM clocks)
__device__ long long g_dbg_ts[1024 * 16];
#define SHARQ_TS(i) do { if ((threadIdx.x & 31) == 0 && blockIdx.x < 1024) g_dbg_ts[blockIdx.x * 16 + (i)] = clock64(); } while (0)
#else
#define SHARQ_TS(i) do { } while (0)
#endif
constexpr int kTmemCols = 512;

// Grouped (MoE) launches: the expert table is built by every CTA in its own shared memory from the DEVICE array
// `offsets` (no host copy of the routing result, no device -> host synchronisation after the router):
// offs[e] = offsets[e], pref[e] = first 128-row block of expert e in the padded row numbering.
struct GroupTab {
  const int32_t* offs;                     // shared memory, E + 1 entries (nullptr: single problem)
  const int32_t* pref;                     // shared memory, E + 1 entries
  int32_t E;
};

struct KParams {
  const uint8_t *sp_sf, *sp_meta, *dn_sf, *w_sf_sp, *w_sf_dn;
  const float *row_scale, *w_ts;
  const uint16_t* bias;
  void* Y;
  int64_t ldy;
  int32_t T, D, K, out_fp32, path;
  int32_t m_blocks, total_tiles;   // grouped: m_blocks = capacity of the activation buffers in 128-row blocks, and
                                   // both are replaced inside the kernel by the values the expert table gives
  const int32_t* offsets;          // grouped: device int32[E + 1] (nullptr otherwise)
  int32_t E;
  // Table 5 combinations (path 3 = dense + dense, 4 = sparse + sparse): the tile runs the K-loop twice
  // into the same accumulator, the second time on the SECOND operand of the same kind (tensor map tm_alt, scale
  // factors sf2, metadata meta2); W is streamed twice
  const uint8_t *sf2, *meta2;
  int32_t group_m;    // pair kernel: 256-row blocks per supertile (tile order, see pair_tile)
  int32_t a_rows;     // rows of the activation TMA boxes: 128, or roundup(T, 8) when T < 128 (out-of-bounds
                      // rows are zero-filled slowly; rows beyond the box keep stale smem, which only feeds
                      // accumulator rows that are never stored)
};

// ---- shared-memory stage layout -------------------------------------------------------------
// SPLIT = the split-K variant for T <= 256 (few output tiles): a thread-block cluster of `splits` CTAs
// shares one output tile, each CTA runs a slice of K, the partial accumulators are exchanged through
// distributed shared memory (16-column slices, owner = slice % splits) and summed in rank order.
// AR = rows reserved for the activation tiles (16 / 64 / 128): for T < 128 only roundup(T, 8) rows are loaded,
// and a smaller reservation leaves room for more ring stages, i.e. more weight bytes in flight per SM (the
// decode shapes are bound by exactly that).  The MMA still reads 128 rows; rows beyond the loaded ones are
// whatever follows in shared memory and only reach accumulator rows that are never stored.
// sharq_prepare_linear (N2): shared memory of the in-kernel sharq_prepare rows (prepare_rows' layout for up to 16
// warps with gamma staged) and the widest row the fused kernel takes
constexpr int kPrepWarpsMax = 16;                 // K <= 16384
constexpr int kPrepSmem = kPrepWarpsMax * 1024 + 256 + 16 + 64 + kPrepWarpsMax * 32 * 64 + 128;

template <int BN, int FMT, bool SPLIT, int AR, int EXTRA = 0>
struct Stage {
  static constexpr int NB = (BN + 127) / 128;                         // 128-row scale atoms of W per tile
  static constexpr int SF_DN_BYTES = (FMT == SHARQ_NVFP4) ? 2048 : 1024;  // per 128 rows per k-block
  static constexpr int A_DN_BYTES = AR * 128 < 1024 ? 1024 : AR * 128;
  static constexpr int A_SP_BYTES = AR * 64 < 1024 ? 1024 : AR * 64;
  static constexpr int A_DN = 0;
  static constexpr int W = A_DN + A_DN_BYTES;
  static constexpr int A_SP = W + BN * 128;
  static constexpr int META = A_SP + A_SP_BYTES;
  static constexpr int SFA_SP = META + 2048;
  static constexpr int SFA_DN = SFA_SP + 1024;
  static constexpr int SFB_SP = SFA_DN + SF_DN_BYTES;
  static constexpr int SFB_DN = SFB_SP + NB * 1024;
  static constexpr int RAW = SFB_DN + NB * SF_DN_BYTES;
  static constexpr int BYTES = (RAW + 1023) / 1024 * 1024;
  static constexpr int NSL = BN / 16;                                 // 16-column slices of the accumulator
  static constexpr int RECV = SPLIT ? (NSL + 2) * AR * 64 : 0;        // [src][slot][AR rows][16 fp32]; S*ceil(NSL/S) <= NSL+2 for S in {2,3,4,8}
  static constexpr int PAD = AR < 128 ? 128 * 128 : 0;               // the MMA's over-read behind the last stage
  static constexpr int GRP = (!SPLIT && AR == 128 && (BN == 128 || BN == 192)) ? 2 * (kMaxExperts + 1) * 4 + 8 : 0;   // expert table (grouped)
  static constexpr int STG = SPLIT ? 0 : kStageBytes;                  // epilogue staging (persistent variants)
  static constexpr int FIT = (232448 - 1024 - 256 - RECV - PAD - GRP - EXTRA - STG) / BYTES;
  static constexpr int STAGES = FIT > 8 ? 8 : FIT;
  static constexpr int SMEM = STAGES * BYTES + PAD + RECV + 1024 /*alignment slack*/ + 256 /*barriers*/ + GRP + EXTRA + STG;
  // tensor-memory columns: two accumulator stages, then metadata and scale factors
  static constexpr int SFB_COLS = NB * 4;          // columns one MMA's B scales occupy
  static constexpr int ACC_STAGES = 2 * BN + 76 <= 512 ? 2 : 1;      // 128- and 192-wide tiles: drain overlaps the next tile
  static constexpr int E_COL = BN * ACC_STAGES > 256 ? BN * ACC_STAGES : 256;   // first column after the accumulators
  static constexpr int SFA_SP_COL = E_COL + 4;     // 2 MMAs x 4
  static constexpr int SFA_DN_COL = E_COL + 12;    // 4 MMAs x 4
  static constexpr int SFB_SP_COL = E_COL + 28;    // 2 MMAs x SFB_COLS (<= 16)
  static constexpr int SFB_DN_COL = E_COL + 44;    // 4 MMAs x SFB_COLS (<= 32)
  static_assert(SFB_DN_COL + 32 <= 512, "tensor memory");
  static_assert(STAGES >= 2, "shared memory: fewer than two ring stages");
};

struct Unit { int m_blk, n_blk, expert, rows_valid, kb0, kb1; };

__device__ __forceinline__ Unit decode_unit(const KParams& p, const GroupTab& g, int m_blocks, int total_tiles,
                                            int tile, int rank, int splits) {
  Unit u;
  if (g.E > 0) {                                   // experts: n fastest, so concurrent CTAs share one expert's
    const int n_tiles = total_tiles / m_blocks;    // A block and weights instead of streaming 50 experts at once
    u.n_blk = tile % n_tiles;
    u.m_blk = tile / n_tiles;
  } else {
    u.m_blk = tile % m_blocks;                     // m fastest: concurrent CTAs share W tiles in L2
    u.n_blk = tile / m_blocks;
  }
  u.expert = 0;
  if (g.E > 0) {
    int lo = 0, hi = g.E - 1;                      // last expert whose first block is <= m_blk (binary search)
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (g.pref[mid] <= u.m_blk) lo = mid; else hi = mid - 1;
    }
    u.expert = lo;
    u.rows_valid = min(BM, (g.offs[lo + 1] - g.offs[lo]) - (u.m_blk - g.pref[lo]) * BM);
  } else {
    u.rows_valid = min(BM, p.T - u.m_blk * BM);
  }
  const int num_kb = (p.K / BK) * (p.path >= 3 ? 2 : 1);   // combinations: second pass = k-blocks num_kb .. 2 num_kb - 1
  u.kb0 = (int)((int64_t)rank * num_kb / splits);
  u.kb1 = (int)((int64_t)(rank + 1) * num_kb / splits);
  return u;
}

// y = acc * scale (+ bias) for N consecutive output features of one row, bf16 or fp32 store.  Columns at or beyond D
// (the ragged last n-tile: D % 8 == 0, any multiple of 8) are neither computed with bias nor stored.
template <int N>
__device__ __forceinline__ void store_row(const KParams& p, int64_t row, int col0, float scale, float (&f)[N]) {
  const int ncols = p.D - col0;                       // >= N for every tile but a ragged last one
  if (ncols <= 0) return;
#pragma unroll
  for (int i = 0; i < N; ++i) f[i] = __fmul_rn(f[i], scale);
  if (ncols >= N) {                                   // the common case, no per-column predicates
    if (p.bias) {
      const uint16_t* b = p.bias + col0;
#pragma unroll
      for (int i = 0; i < N; ++i) f[i] = __fadd_rn(f[i], __uint_as_float((uint32_t)b[i] << 16));
    }
    if (p.out_fp32) {
      float4* dst = reinterpret_cast<float4*>(static_cast<float*>(p.Y) + row * p.ldy + col0);
#pragma unroll
      for (int i = 0; i < N / 4; ++i) dst[i] = make_float4(f[4 * i], f[4 * i + 1], f[4 * i + 2], f[4 * i + 3]);
    } else {
      uint4* dst = reinterpret_cast<uint4*>(static_cast<uint16_t*>(p.Y) + row * p.ldy + col0);
#pragma unroll
      for (int i = 0; i < N / 8; ++i)
        dst[i] = make_uint4(pack_bf16x2_rn(f[8 * i], f[8 * i + 1]), pack_bf16x2_rn(f[8 * i + 2], f[8 * i + 3]),
                            pack_bf16x2_rn(f[8 * i + 4], f[8 * i + 5]), pack_bf16x2_rn(f[8 * i + 6], f[8 * i + 7]));
    }
    return;
  }
  if (p.bias) {
    const uint16_t* b = p.bias + col0;
#pragma unroll
    for (int i = 0; i < N; ++i)
      if (i < ncols) f[i] = __fadd_rn(f[i], __uint_as_float((uint32_t)b[i] << 16));
  }
  if (p.out_fp32) {
    float4* dst = reinterpret_cast<float4*>(static_cast<float*>(p.Y) + row * p.ldy + col0);
#pragma unroll
    for (int i = 0; i < N / 4; ++i)
      if (4 * i < ncols) dst[i] = make_float4(f[4 * i], f[4 * i + 1], f[4 * i + 2], f[4 * i + 3]);
  } else {
    uint4* dst = reinterpret_cast<uint4*>(static_cast<uint16_t*>(p.Y) + row * p.ldy + col0);
#pragma unroll
    for (int i = 0; i < N / 8; ++i)
      if (8 * i < ncols)
        dst[i] = make_uint4(pack_bf16x2_rn(f[8 * i], f[8 * i + 1]), pack_bf16x2_rn(f[8 * i + 2], f[8 * i + 3]),
                            pack_bf16x2_rn(f[8 * i + 4], f[8 * i + 5]), pack_bf16x2_rn(f[8 * i + 6], f[8 * i + 7]));
  }
}

// MC = true (grouped GEMM): a cluster of two CTAs works on two neighbouring n-tiles of the same 128-row block in
// lock step; each CTA fetches half of the shared activation operands and multicasts them to both (the many
// short tiles of the expert GEMMs are bound by L2 -> SM traffic, 60 % of which is the activation side).
//
// FUSED = true (sharq_prepare_linear, SURVEY.md 8(f) N2, T <= 8): warps 6 .. of EVERY CTA run sharq_prepare for all T
// rows (prepare_rows on named barrier 2: the row-per-CTA kernel's body, one warp per 1024 elements of a row) while
// warp 0 already streams the weights.  Every CTA prepares the rows itself: no cross-CTA wait (an earlier version
// released the producers through a device-scope counter and lost 4-6 us waiting for the last CTA to be scheduled).
// The prepared operands go to the caller's activation buffers in global memory -- all CTAs write the same bytes --
// and come back through the same TMA loads as in the two-launch path, after this CTA's own stores are fenced
// (__threadfence + fence.proxy.async) and its `act_bar` mbarrier has completed.
// COMBO = true: the Table 5 combinations (path 3 / 4): second K-loop on the second operand (tm_alt, sf2, meta2).
// The body is shared; the __global__ wrappers below differ in their parameter lists, so that the plain kernel --
// every decode and MoE launch -- carries neither the fourth tensor map nor the prepare parameters.
template <int BN, int FMT, bool SPLIT, int AR, int MC, bool FUSED, bool COMBO>
__device__ __forceinline__ void linear_body(const CUtensorMap* tm_a_sp_p, const CUtensorMap* tm_a_dn_p,
                                            const CUtensorMap* tm_w_p, const CUtensorMap* tm_alt_p, const KParams& p,
                                            const PrepParams* pp_p, const int prep_norm) {
  using S = Stage<BN, FMT, SPLIT, AR, FUSED ? kPrepSmem : (MC == 2 ? kStageBytes : 0)>;   // MC == 2: staging for 8 epilogue warps
  static_assert(!(FUSED && MC), "the fused kernel is for single-problem launches");
  static_assert(!(COMBO && (SPLIT || MC || FUSED)), "combinations run on the persistent single-problem variant");
  constexpr bool NV = (FMT == SHARQ_NVFP4);
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t recv_base = smem_base + S::STAGES * S::BYTES + S::PAD;
  const uint32_t bars = recv_base + S::RECV;      // full[STAGES], empty[STAGES], tmem_full[2], tmem_empty[2], ptr
  auto full_bar = [&](int s) { return bars + 8u * s; };
  auto empty_bar = [&](int s) { return bars + 8u * (S::STAGES + s); };
  auto tmem_full_bar = [&](int a) { return bars + 8u * (2 * S::STAGES + a); };
  auto tmem_empty_bar = [&](int a) { return bars + 8u * (2 * S::STAGES + 2 + a); };
  const uint32_t tmem_ptr_smem = bars + 8u * (2 * S::STAGES + 4);
  const uint32_t act_bar = bars + 8u * (2 * S::STAGES + 5);          // FUSED: this CTA's prepared operands are in memory
  int32_t* grp_tab = reinterpret_cast<int32_t*>(smem_raw + (bars + 256u - smem_u32(smem_raw)));   // offs[E+1], pref[E+1]
  uint8_t* prep_smem = smem_raw + (bars + 256u + (uint32_t)S::GRP - smem_u32(smem_raw));          // FUSED: prepare_rows' scratch
  const uint32_t stg_base = bars + 256u + (uint32_t)S::GRP + (FUSED ? (uint32_t)kPrepSmem : 0u);     // epilogue staging (MC == 2: EXTRA + STG)

  // MC == 2 (320 threads; the short-K expert GEMMs are bound by draining and storing the tiles): eight epilogue warps,
  // two per tensor-memory sub-partition, each taking half of the tile's columns; their staging costs a pipeline stage
  // (3 instead of 4), which tiles of <= 4 k-blocks do not miss.  Long-K launches keep MC == 1: four warps, 4 stages.
  constexpr int kEpiWarps = MC == 2 ? 8 : 4;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == 0) SHARQ_TS(0);
  const bool do_sp = p.path == 0 || p.path == 1 || p.path == 4, do_dn = p.path == 0 || p.path == 2 || p.path == 3;
  // work distribution: SPLIT -> one tile per cluster, this CTA's k-slice; else persistent round-robin
  static_assert(!(SPLIT && MC), "split-K clusters and multicast clusters are separate variants");
  const int crank = (SPLIT || MC) ? (int)tc::cluster_ctarank() : 0;
  const int rank = SPLIT ? crank : 0;                  // k-slice owner (split-K only)
  const int splits = SPLIT ? (int)tc::cluster_nctarank() : 1;
  const int tile0 = SPLIT ? (int)tc::cluster_id_x() : MC ? 2 * (int)tc::cluster_id_x() + crank : (int)blockIdx.x;
  int m_blocks = p.m_blocks, total_tiles = p.total_tiles;
  GroupTab g{nullptr, nullptr, 0};

  if (warp == 0 && lane == 0) {
    tc::prefetch_tmap(tm_a_sp_p);
    tc::prefetch_tmap(tm_a_dn_p);
    tc::prefetch_tmap(tm_w_p);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < S::STAGES; ++s) {
      tc::mbar_init(full_bar(s), 1);
      tc::mbar_init(empty_bar(s), MC ? 2 : 1);      // MC: both CTAs of the cluster must have consumed the slot
    }
    for (int a = 0; a < 2; ++a) {
      tc::mbar_init(tmem_full_bar(a), 1);
      tc::mbar_init(tmem_empty_bar(a), kEpiWarps);  // one arrival per epilogue warp
    }
    if constexpr (FUSED) tc::mbar_init(act_bar, 1);
    tc::fence_mbar_init();
  }
  if (warp == 2) tc::tmem_alloc<kTmemCols>(tmem_ptr_smem);
  tc::tc_fence_before();
  if constexpr (MC) {
    __syncwarp();
    tc::cluster_sync_all();                          // the peer's barriers exist before anything is sent to them
  } else {
    __syncthreads();
  }
  tc::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_smem));
  tc::grid_launch_dependents();                          // the next kernel may start its own prologue
  if (warp == 0) SHARQ_TS(1);
  bool dep_synced = false;
  if constexpr (S::GRP > 0) {
    if (p.E > 0) {
      // expert table from the DEVICE offsets (they may be the router's output: wait for the preceding kernel).
      // Every CTA builds its own copy: E + 1 loads, one warp scan.
      tc::grid_dependency_wait();
      dep_synced = true;
      int32_t* offs = grp_tab;
      int32_t* pref = grp_tab + (kMaxExperts + 1);
      for (int i = threadIdx.x; i <= p.E; i += kThreads) offs[i] = p.offsets[i];
      __syncthreads();
      if (warp == 0) {
        const int per = (p.E + 31) / 32;               // lane l scans experts [l * per, l * per + per)
        int sum = 0;
        for (int i = 0; i < per; ++i) {
          const int e = lane * per + i;
          if (e < p.E) sum += (max(offs[e + 1] - offs[e], 0) + BM - 1) / BM;
        }
        int incl = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const int t = __shfl_up_sync(0xffffffffu, incl, d);
          if (lane >= d) incl += t;
        }
        int run = incl - sum;
        for (int i = 0; i < per; ++i) {
          const int e = lane * per + i;
          if (e < p.E) {
            pref[e] = run;
            run += (max(offs[e + 1] - offs[e], 0) + BM - 1) / BM;
          }
        }
        if (lane == 31) pref[p.E] = incl;
      }
      __syncthreads();
      g.offs = offs; g.pref = pref; g.E = p.E;
      const int n_tiles = p.total_tiles;               // grouped: the host passes the n-tiles per row block here
      m_blocks = min(pref[p.E], p.m_blocks);           // never beyond the caller's buffers
      total_tiles = m_blocks * n_tiles;
    }
  }
  const int tile_step = SPLIT ? total_tiles : (int)gridDim.x;

  float split_scale = 0.0f;
  if (warp == 0) {
    // =========================== TMA producer ===============================================
    {
      const bool lead = tc::elect_one() != 0;          // whole warp runs the loop, one lane issues
      const uint64_t pol_act = SPLIT ? tc::policy_evict_last() : tc::policy_evict_normal();
      const uint64_t pol_w = SPLIT ? tc::policy_evict_first() : tc::policy_evict_normal();
      const int64_t Kc = p.K;
      // W codes + W's scales.  MXFP4: the dense view IS the sparse view, one load feeds both paths.  NVFP4: the dense
      // view (every sparse-view scale repeated, P:130 / R7) is read as its own tensor: expanding it from the sparse
      // atoms in shared memory (tried in the MMA warp: LDS / PRMT / STS + fence.proxy.async per k-block) saved 5 % of
      // the DRAM bytes and cost 1-2 us per decode launch, whose k-block issue sequence is the critical path.
      constexpr bool kSharedSfb = !NV;
      uint32_t tx = BN * 128;
      if (do_sp || (kSharedSfb && do_dn)) tx += S::NB * 1024;
      if (do_sp) tx += p.a_rows * 64 + 2048 + 1024;
      if (do_dn) tx += p.a_rows * 128 + S::SF_DN_BYTES + (kSharedSfb ? 0 : S::NB * S::SF_DN_BYTES);
      uint32_t it = 0;                                   // k-blocks issued so far (ring position)
      for (int tile = tile0; tile < total_tiles; tile += tile_step) {
        const Unit u = decode_unit(p, g, m_blocks, total_tiles, tile, rank, splits);
        const int w_row0 = u.expert * p.D + u.n_blk * BN;
        const int64_t wblk0 = w_row0 / 128;
        const uint8_t* sfa_sp = p.sp_sf + (size_t)u.m_blk * (Kc / 128) * 512;
        const uint8_t* sfa_dn = p.dn_sf + (size_t)u.m_blk * (Kc / 256) * (S::SF_DN_BYTES);
        const uint8_t* meta = p.sp_meta + (size_t)u.m_blk * (Kc / 256) * 2048;
        // weight side of k-block kb (codes + both scale views): independent of the preceding kernel
        const int nkb = (int)(Kc / BK);
        auto load_w = [&](int kbv, uint32_t st, uint32_t fb) {
          const int kb = (COMBO && kbv >= nkb) ? kbv - nkb : kbv;   // second pass of a combination: the same W k-blocks again
          if (lead) tc::tma_load_2d(st + S::W, tm_w_p, fb, kb * 128, w_row0, pol_w);
          for (int nb = 0; nb < S::NB; ++nb) {
            if ((do_sp || (kSharedSfb && do_dn)) && lead)
              tc::bulk_load(st + S::SFB_SP + nb * 1024,
                            p.w_sf_sp + ((size_t)(wblk0 + nb) * (Kc / 128) + (size_t)kb * 2) * 512, 1024, fb, pol_w);
            if (!kSharedSfb && do_dn && lead)
              tc::bulk_load(st + S::SFB_DN + nb * S::SF_DN_BYTES,
                            p.w_sf_dn + ((size_t)(wblk0 + nb) * (Kc / 256) + (size_t)kb) * S::SF_DN_BYTES,
                            S::SF_DN_BYTES, fb, pol_w);
          }
        };
        // activation side: written by sharq_prepare, only after griddepcontrol.wait
        auto load_a = [&](int kbv, uint32_t st, uint32_t fb) {
          const bool alt = COMBO && kbv >= nkb;          // combinations: the second operand
          const int kb = alt ? kbv - nkb : kbv;
          if constexpr (MC) {
            // same 128-row block in both CTAs: CTA 0 fetches the dense side, CTA 1 the sparse side, for both
            if (do_sp && crank == 1) {
              if (lead) tc::tma_load_2d_mc(st + S::A_SP, tm_a_sp_p, fb, kb * 64, u.m_blk * BM, 3, pol_act);
              if (lead) tc::bulk_load_mc(st + S::META, meta + (size_t)kb * 2048, 2048, fb, 3, pol_act);
              if (lead) tc::bulk_load_mc(st + S::SFA_SP, sfa_sp + (size_t)kb * 1024, 1024, fb, 3, pol_act);
            }
            if (do_dn && crank == 0) {
              if (lead) tc::tma_load_2d_mc(st + S::A_DN, tm_a_dn_p, fb, kb * 128, u.m_blk * BM, 3, pol_act);
              if (lead) tc::bulk_load_mc(st + S::SFA_DN, sfa_dn + (size_t)kb * S::SF_DN_BYTES, S::SF_DN_BYTES, fb, 3, pol_act);
            }
            return;
          }
          if (!COMBO || !alt) {                          // SharQ and the single-path modes: everything but a combination's second pass
            if (do_sp) {
              if (lead) tc::tma_load_2d(st + S::A_SP, tm_a_sp_p, fb, kb * 64, u.m_blk * BM, pol_act);
              if (lead) tc::bulk_load(st + S::META, meta + (size_t)kb * 2048, 2048, fb, pol_act);
              if (lead) tc::bulk_load(st + S::SFA_SP, sfa_sp + (size_t)kb * 1024, 1024, fb, pol_act);
            }
            if (do_dn) {
              if (lead) tc::tma_load_2d(st + S::A_DN, tm_a_dn_p, fb, kb * 128, u.m_blk * BM, pol_act);
              if (lead) tc::bulk_load(st + S::SFA_DN, sfa_dn + (size_t)kb * S::SF_DN_BYTES, S::SF_DN_BYTES, fb, pol_act);
            }
            return;
          }
          if (do_sp) {
            const size_t mo = (size_t)u.m_blk * (Kc / 256) * 2048 + (size_t)kb * 2048;
            const size_t so = (size_t)u.m_blk * (Kc / 128) * 512 + (size_t)kb * 1024;
            if (lead) tc::tma_load_2d(st + S::A_SP, tm_alt_p, fb, kb * 64, u.m_blk * BM, pol_act);
            if (lead) tc::bulk_load(st + S::META, p.meta2 + mo, 2048, fb, pol_act);
            if (lead) tc::bulk_load(st + S::SFA_SP, p.sf2 + so, 1024, fb, pol_act);
          }
          if (do_dn) {
            const size_t so = ((size_t)u.m_blk * (Kc / 256) + (size_t)kb) * S::SF_DN_BYTES;
            if (lead) tc::tma_load_2d(st + S::A_DN, tm_alt_p, fb, kb * 128, u.m_blk * BM, pol_act);
            if (lead) tc::bulk_load(st + S::SFA_DN, p.sf2 + so, S::SF_DN_BYTES, fb, pol_act);
          }
        };
        int kb = u.kb0;
        if (!dep_synced) {
          // programmatic dependent launch: stream the first STAGES weight k-blocks while the kernel that
          // produces the activations (sharq_prepare) is still finishing, then wait for it
          const int n_early = min(S::STAGES, u.kb1 - u.kb0);
          for (int i = 0; i < n_early; ++i) {
            if (lead) tc::mbar_expect_tx(full_bar(i), tx);
            load_w(kb + i, smem_base + i * S::BYTES, full_bar(i));
          }
          SHARQ_TS(2);
          tc::grid_dependency_wait();
          if constexpr (FUSED) {                         // the rows prepared by this CTA's own warps 6 .. are in memory
            tc::mbar_wait(act_bar, 0);
            asm volatile("fence.proxy.async;" ::: "memory");
          }
          SHARQ_TS(3);
          dep_synced = true;
          for (int i = 0; i < n_early; ++i) load_a(kb + i, smem_base + i * S::BYTES, full_bar(i));
          kb += n_early;
          it += n_early;
        }
        for (; kb < u.kb1; ++kb, ++it) {
          const int s = it % S::STAGES;
          const uint32_t ph = (it / S::STAGES) & 1;
          tc::mbar_wait(empty_bar(s), ph ^ 1);
          const uint32_t st = smem_base + s * S::BYTES;
          const uint32_t fb = full_bar(s);
          if (lead) tc::mbar_expect_tx(fb, tx);
          load_w(kb, st, fb);
          load_a(kb, st, fb);
        }
      }
      if (!dep_synced) tc::grid_dependency_wait();
    }
  } else if (warp == 1) {
    // =========================== MMA issuer =================================================
    {
      const bool lead = tc::elect_one() != 0;
      const uint32_t idesc_sp = tc::idesc_fp4(BM, BN, true, !NV, 0, 0);
      uint32_t it = 0, n_unit = 0;
      for (int tile = tile0; tile < total_tiles; tile += tile_step, ++n_unit) {
        const Unit u = decode_unit(p, g, m_blocks, total_tiles, tile, rank, splits);
        const uint32_t sfb_shift = (uint32_t)(((u.n_blk * BN) % 128) / 32);   // tiles that start inside a 128-row scale atom
        const uint32_t as = n_unit % S::ACC_STAGES;                       // accumulator stage
        const uint32_t acc = tmem_base + as * BN;
        tc::mbar_wait(tmem_empty_bar(as), ((n_unit / S::ACC_STAGES) & 1u) ^ 1u);   // epilogue has drained this stage
        tc::tc_fence_after();
        uint32_t accumulate = 0;
        for (int kb = u.kb0; kb < u.kb1; ++kb, ++it) {
          const int s = it % S::STAGES;
          const uint32_t ph = (it / S::STAGES) & 1;
          tc::mbar_wait(full_bar(s), ph);
          if (it == 0) SHARQ_TS(4);
          if (kb == u.kb1 - 1) SHARQ_TS(5);
          tc::tc_fence_after();
          const uint32_t st = smem_base + s * S::BYTES;
          if (do_sp) {
            if (lead) tc::tc_cp_meta(tmem_base + S::E_COL, tc::smem_desc(st + S::META, 128, 0));
#pragma unroll
            for (int a = 0; a < 2; ++a) {
              if (lead) tc::tc_cp_sf(tmem_base + S::SFA_SP_COL + 4 * a, tc::smem_desc(st + S::SFA_SP + 512 * a, 128, 0));
#pragma unroll
              for (int nb = 0; nb < S::NB; ++nb)
                if (lead) tc::tc_cp_sf(tmem_base + S::SFB_SP_COL + S::SFB_COLS * a + 4 * nb,
                             tc::smem_desc(st + S::SFB_SP + nb * 1024 + 512 * a, 128, 0));
            }
#pragma unroll
            for (int j = 0; j < 2; ++j) {
              if (lead) tc::mma_sparse(acc, tc::smem_desc(st + S::A_SP + 32 * j, 512, 4),
                             tc::smem_desc(st + S::W + 64 * j, 1024, 2), idesc_sp, tmem_base + S::SFA_SP_COL + 4 * j,
                             tmem_base + S::SFB_SP_COL + S::SFB_COLS * j + sfb_shift, tmem_base + S::E_COL + 2 * j,
                             accumulate);
              accumulate = 1;
            }
          }
          if (do_dn) {
            constexpr int ATOMS = NV ? 4 : 2;
#pragma unroll
            for (int a = 0; a < ATOMS; ++a) {
              if (lead) tc::tc_cp_sf(tmem_base + S::SFA_DN_COL + 4 * a, tc::smem_desc(st + S::SFA_DN + 512 * a, 128, 0));
#pragma unroll
              for (int nb = 0; nb < S::NB; ++nb)      // MXFP4: the dense view IS the sparse view (same atoms)
                if (lead) tc::tc_cp_sf(tmem_base + S::SFB_DN_COL + S::SFB_COLS * a + 4 * nb,
                             tc::smem_desc(st + (NV ? S::SFB_DN + nb * S::SF_DN_BYTES : S::SFB_SP + nb * 1024) + 512 * a, 128, 0));
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              const int atom = NV ? j : j / 2;               // MXFP4: two K=64 MMAs share one 4-scale atom
              const uint32_t sf_id = NV ? 0u : (uint32_t)(j & 1) * 2u;
              const uint32_t idesc_dn = tc::idesc_fp4(BM, BN, false, !NV, sf_id, sf_id);
              if (lead) tc::mma_dense<NV>(acc, tc::smem_desc(st + S::A_DN + 32 * j, 1024, 2),
                                tc::smem_desc(st + S::W + 32 * j, 1024, 2), idesc_dn,
                                tmem_base + S::SFA_DN_COL + 4 * atom,
                                tmem_base + S::SFB_DN_COL + S::SFB_COLS * atom + sfb_shift, accumulate);
              accumulate = 1;
            }
          }
          if constexpr (MC) {
            if (lead) tc::tc_commit_mc(empty_bar(s), 3);           // ... in BOTH CTAs: either may refill the other's slot
          } else {
            if (lead) tc::tc_commit(empty_bar(s));                 // smem slot reusable once these MMAs have read it
          }
        }
        if (lead) tc::tc_commit(tmem_full_bar(as));                // accumulator complete
      }
    }
  } else if (warp < 2 + kEpiWarps) {
    // =========================== epilogue ====================================================
    tc::grid_dependency_wait();                          // row_scale is sharq_prepare's; Y may still be read
    if constexpr (FUSED) tc::mbar_wait(act_bar, 0);      // ... here: this launch's own prepare warps write it
    const int sub = warp & 3;                            // TMEM sub-partition this warp may read
    const int r_local = sub * 32 + lane;
    const uint32_t lane_addr = tmem_base + ((uint32_t)(sub * 32) << 16);
    if constexpr (!SPLIT) {
      uint32_t n_unit = 0;
      const bool one_shot = total_tiles <= tile_step;      // every CTA drains at most one tile (decode launches)
      for (int tile = tile0; tile < total_tiles; tile += tile_step, ++n_unit) {
        const Unit u = decode_unit(p, g, m_blocks, total_tiles, tile, 0, 1);
        const uint32_t as = n_unit % S::ACC_STAGES;
        const int64_t row = (int64_t)u.m_blk * BM + r_local;
        const bool row_ok = r_local < u.rows_valid;
        const float scale = row_ok ? __fmul_rn(FUSED ? __ldcg(p.row_scale + row) : p.row_scale[row], p.w_ts[u.expert]) : 0.0f;
        tc::mbar_wait(tmem_full_bar(as), (n_unit / S::ACC_STAGES) & 1u);
        tc::tc_fence_after();
        if constexpr (MC == 2) {
          const int half = (warp - 2) >> 2;                // columns [half BN / 2, (half + 1) BN / 2)
          epilogue_tile<BN / 2>(p, lane_addr + as * BN + half * (BN / 2), stg_base + (uint32_t)(sub + 4 * half) * 4096u, lane,
                                (int64_t)u.m_blk * BM + sub * 32, min(32, max(0, u.rows_valid - sub * 32)),
                                u.n_blk * BN + half * (BN / 2), scale);
        } else if (one_shot) {
          epilogue_tile<BN, false>(p, lane_addr + as * BN, stg_base + (uint32_t)sub * 4096u, lane, (int64_t)u.m_blk * BM + sub * 32,
                                   min(32, max(0, u.rows_valid - sub * 32)), u.n_blk * BN, scale);
        } else {
          epilogue_tile<BN>(p, lane_addr + as * BN, stg_base + (uint32_t)sub * 4096u, lane, (int64_t)u.m_blk * BM + sub * 32,
                            min(32, max(0, u.rows_valid - sub * 32)), u.n_blk * BN, scale);
        }
        tc::tc_fence_before();
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(tmem_empty_bar(as));
      }
    } else {
      // ---- split-K: scatter 16-column slices of the partial accumulator to their owner CTAs ----
      const Unit u = decode_unit(p, g, m_blocks, total_tiles, tile0, rank, splits);
      const bool row_ok = r_local < u.rows_valid;
      const int slots = (BN / 16 + splits - 1) / splits;
      // the output scale of this thread's row, fetched while the main loop runs (used after the exchange)
      if (row_ok) {
        const float* rs = p.row_scale + (int64_t)u.m_blk * BM + r_local;
        split_scale = __fmul_rn(FUSED ? __ldcg(rs) : *rs, p.w_ts[u.expert]);
      }
      tc::mbar_wait(tmem_full_bar(0), 0);
      if (warp == 2) SHARQ_TS(6);
      tc::tc_fence_after();
#pragma unroll 1
      for (int j4 = 0; j4 < BN / 64; ++j4) {              // four 16-column slices (two tensor-memory loads) in flight
        uint32_t v[64];
        tc::tmem_ld32(lane_addr + j4 * 64, *reinterpret_cast<uint32_t(*)[32]>(&v[0]));
        tc::tmem_ld32(lane_addr + j4 * 64 + 32, *reinterpret_cast<uint32_t(*)[32]>(&v[32]));
        tc::tmem_ld_wait();
        if (row_ok) {
          // exchange layout [src][slot][16-byte chunk][row]: the 32 lanes of one store are 512 contiguous
          // bytes (full lines on the SM-to-SM network, no bank conflicts on either side)
#pragma unroll
          for (int h = 0; h < 4; ++h) {
            const int j = 4 * j4 + h;
            const uint32_t local = recv_base + (uint32_t)((rank * slots + j / splits) * AR * 64 + r_local * 16);
            const int owner = j % splits;
            if (owner == rank) {                         // this CTA's own slices never leave its shared memory
#pragma unroll
              for (int i = 0; i < 4; ++i)
                tc::st_shared_v4(local + (uint32_t)(i * AR * 16), __uint_as_float(v[16 * h + 4 * i]),
                                 __uint_as_float(v[16 * h + 4 * i + 1]), __uint_as_float(v[16 * h + 4 * i + 2]),
                                 __uint_as_float(v[16 * h + 4 * i + 3]));
            } else {
              const uint32_t remote = tc::map_to_cta(local, (uint32_t)owner);
#pragma unroll
              for (int i = 0; i < 4; ++i)
                tc::st_cluster_v4(remote + (uint32_t)(i * AR * 16), __uint_as_float(v[16 * h + 4 * i]),
                                  __uint_as_float(v[16 * h + 4 * i + 1]), __uint_as_float(v[16 * h + 4 * i + 2]),
                                  __uint_as_float(v[16 * h + 4 * i + 3]));
            }
          }
        }
      }
      tc::tc_fence_before();
    }
  } else {
    // =========================== in-kernel sharq_prepare (FUSED only: warps 6 ..) ==================
    if constexpr (FUSED) {
      tc::grid_dependency_wait();                        // x belongs to the kernels before this one
      const int ptid = (int)threadIdx.x - kThreads, pthreads = (int)blockDim.x - kThreads;
      if (prep_norm == SHARQ_NORM_RMS) prepare_rows<FMT, SHARQ_NORM_RMS, 2, false>(*pp_p, prep_smem, ptid, pthreads, 0, 1);
#ifdef SHARQ_EXPERIMENTS
      else if (prep_norm == 99) { }                      // timing experiment: no in-kernel prepare at all
#endif
      else prepare_rows<FMT, SHARQ_NORM_NONE, 2, false>(*pp_p, prep_smem, ptid, pthreads, 0, 1);
      __threadfence();                                   // every thread's stores, device scope
      named_bar_sync<2>(pthreads);
      if (ptid == 0) tc::mbar_arrive(act_bar);
    }
  }
  if constexpr (SPLIT) {
    __syncwarp();
    if (warp == 2) SHARQ_TS(7);
    tc::cluster_sync_all();                              // partial slices have landed in their owners
    if (warp == 2) SHARQ_TS(8);
    if (warp >= 2 && warp < 6) {
      const Unit u = decode_unit(p, g, m_blocks, total_tiles, tile0, rank, splits);
      const int r_local = (warp & 3) * 32 + lane;
      if (r_local < u.rows_valid) {
        const int64_t row = (int64_t)u.m_blk * BM + r_local;
        const float scale = split_scale;
        const int slots = (BN / 16 + splits - 1) / splits;
        for (int slot = 0; slot < slots; ++slot) {
          const int j = slot * splits + rank;            // the slices this CTA owns
          if (j >= BN / 16) break;
          float f[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) f[i] = 0.0f;
          for (int s0 = 0; s0 < splits; s0 += 4) {       // fixed order: deterministic sum; four sources' loads in flight
            float4 t[4][4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              if (s0 + q < splits) {
                const uint32_t a = recv_base + (uint32_t)(((s0 + q) * slots + slot) * AR * 64 + r_local * 16);
#pragma unroll
                for (int i = 0; i < 4; ++i) t[q][i] = tc::ld_shared_v4(a + (uint32_t)(i * AR * 16));
              }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              if (s0 + q < splits) {
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                  f[4 * i] = __fadd_rn(f[4 * i], t[q][i].x); f[4 * i + 1] = __fadd_rn(f[4 * i + 1], t[q][i].y);
                  f[4 * i + 2] = __fadd_rn(f[4 * i + 2], t[q][i].z); f[4 * i + 3] = __fadd_rn(f[4 * i + 3], t[q][i].w);
                }
              }
            }
          }
          store_row<16>(p, row, u.n_blk * BN + j * 16, scale, f);
        }
      }
    }
  }
  if constexpr (MC) {
    __syncwarp();
    tc::cluster_sync_all();                              // the peer may still multicast into / signal this CTA
  }
  if (warp == 2) SHARQ_TS(9);
  __syncthreads();
  if (warp == 2) {
    tc::tc_fence_after();
    tc::tmem_dealloc<kTmemCols>(tmem_base);
  }
}

template <int BN, int FMT, bool SPLIT, int AR, int MC = 0>
__global__ void __launch_bounds__(MC == 2 ? kThreads + 128 : kThreads, 1)
sharq_linear_kernel(const __grid_constant__ CUtensorMap tm_a_sp, const __grid_constant__ CUtensorMap tm_a_dn,
                    const __grid_constant__ CUtensorMap tm_w, const KParams p) {
  linear_body<BN, FMT, SPLIT, AR, MC, false, false>(&tm_a_sp, &tm_a_dn, &tm_w, nullptr, p, nullptr, 0);
}

template <int BN, int FMT, int AR>
__global__ void __launch_bounds__(kThreads, 1)
sharq_linear_combo_kernel(const __grid_constant__ CUtensorMap tm_a_sp, const __grid_constant__ CUtensorMap tm_a_dn,
                          const __grid_constant__ CUtensorMap tm_w, const __grid_constant__ CUtensorMap tm_alt,
                          const KParams p) {
  linear_body<BN, FMT, false, AR, false, false, true>(&tm_a_sp, &tm_a_dn, &tm_w, &tm_alt, p, nullptr, 0);
}

template <int BN, int FMT, bool SPLIT, int AR>
__global__ void __launch_bounds__(kThreads + 32 * kPrepWarpsMax, 1)
sharq_linear_fused_kernel(const __grid_constant__ CUtensorMap tm_a_sp, const __grid_constant__ CUtensorMap tm_a_dn,
                          const __grid_constant__ CUtensorMap tm_w, const KParams p,
                          const __grid_constant__ PrepParams pp, const int prep_norm) {
  linear_body<BN, FMT, SPLIT, AR, false, true, false>(&tm_a_sp, &tm_a_dn, &tm_w, nullptr, p, &pp, prep_norm);
}

// ---- CTA-pair kernel (cta_group::2): 256 x 256 output tile per cluster of two CTAs ---------------------
// For T >= 256 the 128 x 128 kernel is bound by shared-memory refill latency (48 KB per 384 MMA cycles).
// Here each CTA stages its own 128 rows of A but only HALF of the 256-row W tile, and one tcgen05.mma
// with M = 256, N = 256 consumes both CTAs' shared memory: same bytes per stage, twice the MMA work.
// PBN = tile width: 192 -> two TMEM accumulator stages (2 x 192 + 76 scale / metadata columns <= 512), so the
// epilogue of tile i overlaps the main loop of tile i+1, and finer wave quantisation; 256 -> one stage.
template <int FMT, int PBN>
struct PairStage {
  static constexpr int SF_DN_BYTES = (FMT == SHARQ_NVFP4) ? 2048 : 1024;
  static constexpr int BN = PBN;
  static constexpr int HALF = PBN / 2;                   // W rows this CTA stages
  static constexpr int A_DN = 0;
  static constexpr int W = A_DN + BM * 128;
  static constexpr int A_SP = W + HALF * 128;
  static constexpr int META = A_SP + BM * 64;
  static constexpr int SFA_SP = META + 2048;
  static constexpr int SFA_DN = SFA_SP + 1024;
  static constexpr int SFB_SP = SFA_DN + SF_DN_BYTES;    // two 128-row atoms rows: both CTAs need every B scale
  static constexpr int SFB_DN = SFB_SP + 2 * 1024;
  static constexpr int RAW = SFB_DN + 2 * SF_DN_BYTES;
  static constexpr int BYTES = (RAW + 1023) / 1024 * 1024;
  static constexpr int STAGES = 4;
  static constexpr int SMEM = STAGES * BYTES + 1024 + 256 + kStageBytes;
  static constexpr int GRP = 3 * (kMaxExperts + 1) * 4 + 16;      // grouped: offs, pair prefix, block prefix per expert
  static constexpr int SMEM_GROUPED = SMEM + GRP;
  static constexpr int ACC_STAGES = PBN <= 192 ? 2 : 1;
  static constexpr int SFB_COLS = 8;
  static constexpr int SF0 = PBN * ACC_STAGES;           // first column after the accumulators
  static constexpr int E_COL = SF0, SFA_SP_COL = SF0 + 4, SFA_DN_COL = SF0 + 12, SFB_SP_COL = SF0 + 28,
                       SFB_DN_COL = SF0 + 44;
  static_assert(SF0 + 76 <= 512, "tensor memory");
};

// One unit of work of the pair kernel: which 128-row block this CTA contributes, which n-tile, how many of its rows
// are real, and (grouped) which expert's weights.
struct PairUnit { int m_blk, n_blk, rows_valid, expert; };

// GROUPED = true (sharq_linear_grouped, MoE experts with more than 128 rows): a pair works on two consecutive 128-row
// blocks of ONE expert (the second block may not exist: its CTA then contributes rows that are never stored) and on
// that expert's weight rows.  Tiles run n-fastest inside a pair, so the clusters running at the same time share a few
// experts' activation blocks (L2) and every weight tile is read from DRAM by exactly one cluster.  The expert table
// (row offsets, prefix of pairs, prefix of 128-row blocks in the padded row numbering) is built by every CTA in its
// own shared memory from the DEVICE array `offsets`.
template <int FMT, int PBN, bool GROUPED = false>
__global__ void __launch_bounds__(kThreads, 1)
sharq_linear_pair_kernel(const __grid_constant__ CUtensorMap tm_a_sp, const __grid_constant__ CUtensorMap tm_a_dn,
                         const __grid_constant__ CUtensorMap tm_w, const __grid_constant__ CUtensorMap tm_sfa_sp,
                         const __grid_constant__ CUtensorMap tm_sfa_dn, const __grid_constant__ CUtensorMap tm_meta,
                         const __grid_constant__ CUtensorMap tm_sfb_sp, const __grid_constant__ CUtensorMap tm_sfb_dn,
                         const KParams p) {
  using S = PairStage<FMT, PBN>;
  constexpr bool NV = (FMT == SHARQ_NVFP4);
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bars = smem_base + S::STAGES * S::BYTES;
  auto full_bar = [&](int s) { return bars + 8u * s; };                       // used in the leader CTA
  auto empty_bar = [&](int s) { return bars + 8u * (2 * S::STAGES + s); };
  auto tmem_full_bar = [&](int a) { return bars + 8u * (3 * S::STAGES + a); };
  auto tmem_empty_bar = [&](int a) { return bars + 8u * (3 * S::STAGES + 2 + a); };   // leader CTA
  const uint32_t tmem_ptr_smem = bars + 8u * (3 * S::STAGES + 4);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rank = (int)tc::cluster_ctarank();
  const bool do_sp = p.path != 2, do_dn = p.path != 1;
  const int num_kb = p.K / BK;
  int m_pairs = (p.m_blocks + 1) / 2;
  const int n_tiles = (p.D + S::BN - 1) / S::BN;                // the last tile may be ragged in N
  const int gm = p.group_m > 0 && p.group_m < m_pairs ? p.group_m : m_pairs;
  const int tile0 = (int)tc::cluster_id_x(), tile_step = (int)(gridDim.x >> 1);
  const uint32_t stg_base = bars + 256u;                                    // epilogue staging, then the grouped tables
  const int32_t* g_offs = reinterpret_cast<const int32_t*>(smem_raw + (bars + 256u + (uint32_t)kStageBytes - smem_u32(smem_raw)));
  const int32_t* g_ppref = g_offs + (kMaxExperts + 1);
  const int32_t* g_bpref = g_ppref + (kMaxExperts + 1);

  if (warp == 0 && lane == 0) {
    tc::prefetch_tmap(&tm_a_sp);
    tc::prefetch_tmap(&tm_a_dn);
    tc::prefetch_tmap(&tm_w);
    tc::prefetch_tmap(&tm_sfa_sp);
    tc::prefetch_tmap(&tm_sfa_dn);
    tc::prefetch_tmap(&tm_meta);
    tc::prefetch_tmap(&tm_sfb_sp);
    tc::prefetch_tmap(&tm_sfb_dn);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < S::STAGES; ++s) {
      tc::mbar_init(full_bar(s), 1);             // leader's expect_tx; every load of the pair completes here
      tc::mbar_init(empty_bar(s), 1);
    }
    for (int a = 0; a < 2; ++a) {
      tc::mbar_init(tmem_full_bar(a), 1);
      tc::mbar_init(tmem_empty_bar(a), 8);       // four epilogue warps in each CTA
    }
    tc::fence_mbar_init();
  }
  if (warp == 2) tc::tmem_alloc_pair<kTmemCols>(tmem_ptr_smem);
  tc::tc_fence_before();
  __syncwarp();
  tc::cluster_sync_all();                        // peer barriers initialised before any remote signal
  tc::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_smem));
  tc::grid_launch_dependents();
  tc::grid_dependency_wait();
  if constexpr (GROUPED) {
    int32_t* offs = const_cast<int32_t*>(g_offs);
    int32_t* ppref = const_cast<int32_t*>(g_ppref);
    int32_t* bpref = const_cast<int32_t*>(g_bpref);
    for (int i = threadIdx.x; i <= p.E; i += kThreads) offs[i] = p.offsets[i];
    __syncthreads();
    if (warp == 0) {
      const int per = (p.E + 31) / 32;                 // lane l scans experts [l * per, l * per + per)
      int sp = 0, sb = 0;
      for (int i = 0; i < per; ++i) {
        const int e = lane * per + i;
        if (e < p.E) {
          const int c = max(offs[e + 1] - offs[e], 0);
          sp += (c + 2 * BM - 1) / (2 * BM);
          sb += (c + BM - 1) / BM;
        }
      }
      int ip = sp, ib = sb;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const int tp = __shfl_up_sync(0xffffffffu, ip, d), tb = __shfl_up_sync(0xffffffffu, ib, d);
        if (lane >= d) { ip += tp; ib += tb; }
      }
      int rp = ip - sp, rb = ib - sb;
      for (int i = 0; i < per; ++i) {
        const int e = lane * per + i;
        if (e < p.E) {
          ppref[e] = rp; bpref[e] = rb;
          const int c = max(offs[e + 1] - offs[e], 0);
          rp += (c + 2 * BM - 1) / (2 * BM);
          rb += (c + BM - 1) / BM;
        }
      }
      if (lane == 31) { ppref[p.E] = ip; bpref[p.E] = ib; }
    }
    __syncthreads();
    m_pairs = g_ppref[p.E];
  }
  const int total = m_pairs * n_tiles;
  auto unit_of = [&](int tile) {
    PairUnit u;
    if constexpr (GROUPED) {
      const int gp = tile / n_tiles;
      u.n_blk = tile - gp * n_tiles;
      int lo = 0, hi = p.E - 1;                        // last expert whose first pair is <= gp
      while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (g_ppref[mid] <= gp) lo = mid; else hi = mid - 1;
      }
      u.expert = lo;
      const int b = 2 * (gp - g_ppref[lo]) + rank;     // this CTA's block inside the expert
      u.m_blk = g_bpref[lo] + b;
      const int left = (g_offs[lo + 1] - g_offs[lo]) - b * BM;
      u.rows_valid = (u.m_blk < p.m_blocks) ? max(0, min(BM, left)) : 0;     // never beyond the caller's buffers
    } else {
      int m_pair;
      pair_tile(tile, m_pairs, n_tiles, gm, m_pair, u.n_blk);
      u.m_blk = 2 * m_pair + rank;
      u.expert = 0;
      u.rows_valid = max(0, min(BM, p.T - u.m_blk * BM));
    }
    return u;
  };

  if (warp == 0) {
    // =========================== TMA producer (both CTAs) ===================================
    {
      const bool lead = tc::elect_one() != 0;
      const uint64_t pol = tc::policy_evict_normal();
      // every load of the pair (tiles, scale-factor atoms, metadata) is a cta_group::2 tensor copy whose
      // complete_tx lands on the LEADER's full barrier: no cross-CTA hand-off inside the ring
      const uint32_t tx = 2u * (S::HALF * 128 + (do_sp ? BM * 64 + 2048 + 1024 + 2 * 1024 : 0) +
                                (do_dn ? BM * 128 + 3 * S::SF_DN_BYTES : 0));
      constexpr int DN_ROWS = S::SF_DN_BYTES / 1024;       // 1024-byte rows of the scale-factor tensor maps
      const int kq = p.K / 256;
      uint32_t it = 0;
      for (int tile = tile0; tile < total; tile += tile_step) {
        const PairUnit u = unit_of(tile);
        const int m_blk = u.m_blk, n_blk = u.n_blk;
        const int m_sf = min(m_blk, p.m_blocks - 1);       // a ragged pair's second CTA: valid memory, unused rows
        const int n0 = u.expert * p.D + n_blk * S::BN;     // first weight row of the tile (stacked experts)
        const int wblk0 = n0 / 128;
        for (int kb = 0; kb < num_kb; ++kb, ++it) {
          const int s = it % S::STAGES;
          const uint32_t ph = (it / S::STAGES) & 1;
          tc::mbar_wait(empty_bar(s), ph ^ 1);
          const uint32_t st = smem_base + s * S::BYTES;
          const uint32_t fb = full_bar(s);
          if (lead && rank == 0) tc::mbar_expect_tx(fb, tx);
          if (lead) tc::tma_load_2d_pair(st + S::W, &tm_w, fb, kb * 128, n0 + rank * S::HALF, pol);
          if (do_sp) {
            if (lead) tc::tma_load_2d_pair(st + S::A_SP, &tm_a_sp, fb, kb * 64, m_blk * BM, pol);
            if (lead) tc::tma_load_2d_pair(st + S::META, &tm_meta, fb, 0, (m_sf * kq + kb) * 2, pol);
            if (lead) tc::tma_load_2d_pair(st + S::SFA_SP, &tm_sfa_sp, fb, 0, m_sf * kq + kb, pol);
            // both CTAs need the B scales of all 256 rows: each fetches one 128-row atom row for both
            if (lead) tc::tma_load_2d_pair_mc(st + S::SFB_SP + rank * 1024, &tm_sfb_sp, fb, 0, (wblk0 + rank) * kq + kb, 3, pol);
          }
          if (do_dn) {
            if (lead) tc::tma_load_2d_pair(st + S::A_DN, &tm_a_dn, fb, kb * 128, m_blk * BM, pol);
            if (lead) tc::tma_load_2d_pair(st + S::SFA_DN, &tm_sfa_dn, fb, 0, (m_sf * kq + kb) * DN_ROWS, pol);
            if (lead) tc::tma_load_2d_pair_mc(st + S::SFB_DN + rank * S::SF_DN_BYTES, &tm_sfb_dn, fb, 0,
                                              ((wblk0 + rank) * kq + kb) * DN_ROWS, 3, pol);
          }
        }
      }
    }
  } else if (warp == 1) {
    if (rank == 0) {
      const bool lead = tc::elect_one() != 0;
      // =========================== MMA issuer (leader CTA) ===================================
      const uint32_t idesc_sp = tc::idesc_fp4(256, S::BN, true, !NV, 0, 0);
      uint32_t it = 0, n_unit = 0;
      for (int tile = tile0; tile < total; tile += tile_step, ++n_unit) {
        const uint32_t as = n_unit % S::ACC_STAGES;
        const uint32_t acc = tmem_base + as * S::BN;
        int n_blk_u;
        if constexpr (GROUPED) {
          n_blk_u = tile % n_tiles;
        } else {
          int m_pair_u;
          pair_tile(tile, m_pairs, n_tiles, gm, m_pair_u, n_blk_u);
        }
        const uint32_t sfb_shift = (uint32_t)(((n_blk_u * S::BN) % 128) / 32);   // tile starts inside a 128-row atom
        tc::mbar_wait(tmem_empty_bar(as), ((n_unit / S::ACC_STAGES) & 1u) ^ 1u);   // both CTAs' epilogues drained it
        tc::tc_fence_after();
        uint32_t accumulate = 0;
        for (int kb = 0; kb < num_kb; ++kb, ++it) {
          const int s = it % S::STAGES;
          tc::mbar_wait(full_bar(s), (it / S::STAGES) & 1);
          tc::tc_fence_after();
          const uint32_t st = smem_base + s * S::BYTES;
          if (do_sp) {
            if (lead) tc::tc_cp_meta_pair(tmem_base + S::E_COL, tc::smem_desc(st + S::META, 128, 0));
#pragma unroll
            for (int a = 0; a < 2; ++a) {
              if (lead) tc::tc_cp_sf_pair(tmem_base + S::SFA_SP_COL + 4 * a, tc::smem_desc(st + S::SFA_SP + 512 * a, 128, 0));
#pragma unroll
              for (int nb = 0; nb < 2; ++nb)
                if (lead) tc::tc_cp_sf_pair(tmem_base + S::SFB_SP_COL + S::SFB_COLS * a + 4 * nb,
                                  tc::smem_desc(st + S::SFB_SP + nb * 1024 + 512 * a, 128, 0));
            }
#pragma unroll
            for (int j = 0; j < 2; ++j) {
              if (lead) tc::mma_sparse_pair(acc, tc::smem_desc(st + S::A_SP + 32 * j, 512, 4),
                                  tc::smem_desc(st + S::W + 64 * j, 1024, 2), idesc_sp,
                                  tmem_base + S::SFA_SP_COL + 4 * j,
                                  tmem_base + S::SFB_SP_COL + S::SFB_COLS * j + sfb_shift,
                                  tmem_base + S::E_COL + 2 * j, accumulate);
              accumulate = 1;
            }
          }
          if (do_dn) {
            constexpr int ATOMS = NV ? 4 : 2;
#pragma unroll
            for (int a = 0; a < ATOMS; ++a) {
              if (lead) tc::tc_cp_sf_pair(tmem_base + S::SFA_DN_COL + 4 * a, tc::smem_desc(st + S::SFA_DN + 512 * a, 128, 0));
#pragma unroll
              for (int nb = 0; nb < 2; ++nb)
                if (lead) tc::tc_cp_sf_pair(tmem_base + S::SFB_DN_COL + S::SFB_COLS * a + 4 * nb,
                                  tc::smem_desc(st + S::SFB_DN + nb * S::SF_DN_BYTES + 512 * a, 128, 0));
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              const int atom = NV ? j : j / 2;
              const uint32_t sf_id = NV ? 0u : (uint32_t)(j & 1) * 2u;
              const uint32_t idesc_dn = tc::idesc_fp4(256, S::BN, false, !NV, sf_id, sf_id);
              if (lead) tc::mma_dense_pair<NV>(acc, tc::smem_desc(st + S::A_DN + 32 * j, 1024, 2),
                                     tc::smem_desc(st + S::W + 32 * j, 1024, 2), idesc_dn,
                                     tmem_base + S::SFA_DN_COL + 4 * atom,
                                     tmem_base + S::SFB_DN_COL + S::SFB_COLS * atom + sfb_shift, accumulate);
              accumulate = 1;
            }
          }
          if (lead) tc::tc_commit_pair(empty_bar(s), 3);              // frees this slot in BOTH CTAs
        }
        if (lead) tc::tc_commit_pair(tmem_full_bar(as), 3);
      }
    }
  } else {
    // =========================== epilogue (both CTAs) ==========================================
    const int sub = warp & 3;
    const int r_local = sub * 32 + lane;
    const uint32_t lane_addr = tmem_base + ((uint32_t)(sub * 32) << 16);
    uint32_t n_unit = 0;
    for (int tile = tile0; tile < total; tile += tile_step, ++n_unit) {
      const PairUnit u = unit_of(tile);
      const int n_blk = u.n_blk;
      const int64_t row = (int64_t)u.m_blk * BM + r_local;
      const bool row_ok = r_local < u.rows_valid;
      const float scale = row_ok ? __fmul_rn(p.row_scale[row], p.w_ts[u.expert]) : 0.0f;
      const uint32_t as = n_unit % S::ACC_STAGES;
      tc::mbar_wait(tmem_full_bar(as), (n_unit / S::ACC_STAGES) & 1u);
      tc::tc_fence_after();
      if (total <= tile_step)                        // one tile per pair in its life (T <= 256): the rolled loop
        epilogue_tile<S::BN, false>(p, lane_addr + as * S::BN, stg_base + (uint32_t)sub * 4096u, lane,
                                    (int64_t)u.m_blk * BM + sub * 32, min(32, max(0, u.rows_valid - sub * 32)), n_blk * S::BN, scale);
      else
        epilogue_tile<S::BN>(p, lane_addr + as * S::BN, stg_base + (uint32_t)sub * 4096u, lane, (int64_t)u.m_blk * BM + sub * 32,
                             min(32, max(0, u.rows_valid - sub * 32)), n_blk * S::BN, scale);
      tc::tc_fence_before();
      __syncwarp();
      if (lane == 0) tc::mbar_arrive_cluster(tc::map_to_cta(tmem_empty_bar(as), 0));
    }
  }
  tc::tc_fence_before();
  __syncwarp();
  tc::cluster_sync_all();                        // the peer may still be reading / being written by the pair MMA
  if (warp == 2) {
    tc::tc_fence_after();
    tc::tmem_dealloc_pair<kTmemCols>(tmem_base);
  }
}

// ---- host: tensor maps + launch ----------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {                       // driver entry point, resolved once (C++11 thread-safe static)
  static const EncodeTiledFn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      f = nullptr;
    return reinterpret_cast<EncodeTiledFn>(f);
  }();
  return fn;
}

// bytes [rows, row_bytes] row-major -> boxes of box_rows x box_bytes, swizzle = box_bytes (64 or 128)
bool make_map(CUtensorMap* m, const void* base, uint64_t rows, uint64_t row_bytes, uint32_t box_bytes,
              uint32_t box_rows) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {row_bytes, rows};
  cuuint64_t strides[1] = {row_bytes};
  cuuint32_t box[2] = {box_bytes, box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUtensorMapSwizzle sw = box_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B;
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Device facts the launcher derives once per (kernel variant, device) and then only reads: "the opt-in shared
// memory size of this kernel is set" and "this many clusters of size c are co-resident".  They are answers of the
// CUDA runtime about the device, not library state: lock-free, filled idempotently (two threads racing compute the
// same value), keyed by the device ordinal, a failed query is not cached.
constexpr int kMaxDevices = 64;
inline cudaError_t set_smem_once(std::atomic<uint64_t>& done, const void* kfn, int smem, int dev) {
  if (dev >= 0 && dev < kMaxDevices && ((done.load(std::memory_order_acquire) >> dev) & 1u)) return cudaSuccess;
  const cudaError_t e = cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess && dev >= 0 && dev < kMaxDevices) done.fetch_or(uint64_t(1) << dev, std::memory_order_release);
  return e;
}

// Number of K-splits (cluster size) for a launch with `tiles` output tiles: only when the tiles alone
// leave most SMs idle, only sizes whose slice exchange fits the receive buffer (2, 3, 4, 8), and only if
// all `tiles` clusters are co-resident in ONE wave (cluster placement is per GPC, so tiles * S <= SMs is
// not enough: cudaOccupancyMaxActiveClusters decides).
template <int BN, int FMT, int AR>
int choose_splits(int64_t tiles, int num_kb, int num_sms, int dev) {
  if (tiles * 2 > num_sms) return 1;
  using S = Stage<BN, FMT, true, AR>;
  static std::atomic<int> max_clusters[kMaxDevices][9];          // 0 = not queried yet (zero-initialised)
  static std::atomic<uint64_t> smem_set{0};
  const int cand[4] = {8, 4, 3, 2};
  for (int c : cand) {
    if (tiles * c > num_sms || num_kb < 2 * c) continue;
    int n = (dev >= 0 && dev < kMaxDevices) ? max_clusters[dev][c].load(std::memory_order_relaxed) : 0;
    if (n == 0) {
      cudaLaunchConfig_t lc{};
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = (unsigned)c; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      lc.gridDim = dim3((unsigned)(c * num_sms)); lc.blockDim = dim3(kThreads); lc.dynamicSmemBytes = S::SMEM;
      lc.attrs = at; lc.numAttrs = 1;
      auto kfn = sharq_linear_kernel<BN, FMT, true, AR>;
      if (set_smem_once(smem_set, (const void*)kfn, S::SMEM, dev) != cudaSuccess) continue;
      if (cudaOccupancyMaxActiveClusters(&n, kfn, &lc) != cudaSuccess || n <= 0) continue;   // not cached: asked again
      if (dev >= 0 && dev < kMaxDevices) max_clusters[dev][c].store(n, std::memory_order_relaxed);
    }
    if (n >= tiles) return c;
  }
  return 1;
}

struct LaunchEnv { int num_sms; int dev; cudaStream_t st; LinearPlan* plan_only; const FusedArgs* fz; };

inline void fill_plan(LinearPlan* pl, int kind, int bn, int ar, int splits, int stages, int64_t tiles, int64_t grid,
                      int cluster) {
  pl->kind = kind; pl->bn = bn; pl->act_rows = ar; pl->splits = splits; pl->stages = stages; pl->tiles = tiles;
  pl->grid = grid; pl->cluster = cluster;
}

template <int BN, int FMT, int AR, bool FUSED>
sharq_status launch_1cta_impl(const LinearArgs& a, const KParams& p, const CUtensorMap& tm_sp,
                              const CUtensorMap& tm_dn, const CUtensorMap& tm_w, const CUtensorMap& tm_alt, int64_t tiles,
                              const LaunchEnv& env) {
  constexpr bool kSplitFits = !(BN == 256 && AR == 128);   // no room for the exchange buffers; never needed there
  constexpr int kExtra = FUSED ? kPrepSmem : 0;
  int splits = 1;
  // (the fused kernel takes the cluster size the plain kernel would: one CTA per SM either way)
  if constexpr (kSplitFits) if (p.E == 0 && p.path < 3) splits = choose_splits<BN, FMT, AR>(tiles, (int)(a.K / BK), env.num_sms, env.dev);
  cudaLaunchConfig_t lc{};
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = debug_env().no_pdl ? 0 : 1;
  lc.attrs = attr;
  lc.numAttrs = 1;
  lc.blockDim = dim3(FUSED ? kThreads + 32 * env.fz->warps : kThreads);
  lc.stream = env.st;
  PrepParams pp{};
  int norm = 0;
  if constexpr (FUSED) { pp = *env.fz->pp; norm = env.fz->norm; if (debug_env().skip_prep) norm = 99; }
  if constexpr (kSplitFits) if (splits > 1) {
    using S = Stage<BN, FMT, true, AR, kExtra>;
    if (env.plan_only) { fill_plan(env.plan_only, FUSED ? 4 : 0, BN, AR, splits, S::STAGES, tiles, tiles * splits, splits); return SHARQ_OK; }
    static std::atomic<uint64_t> smem_set{0};
    lc.gridDim = dim3((unsigned)(tiles * splits));
    lc.dynamicSmemBytes = S::SMEM;
    attr[1].id = cudaLaunchAttributeClusterDimension;
    attr[1].val.clusterDim.x = (unsigned)splits;
    attr[1].val.clusterDim.y = 1;
    attr[1].val.clusterDim.z = 1;
    lc.numAttrs = 2;
    if constexpr (FUSED) {
      auto kfn = sharq_linear_fused_kernel<BN, FMT, true, AR>;
      if (set_smem_once(smem_set, (const void*)kfn, S::SMEM, env.dev) != cudaSuccess) return SHARQ_ECUDA;
      return cudaLaunchKernelEx(&lc, kfn, tm_sp, tm_dn, tm_w, p, pp, norm) == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
    } else {
      auto kfn = sharq_linear_kernel<BN, FMT, true, AR>;
      if (set_smem_once(smem_set, (const void*)kfn, S::SMEM, env.dev) != cudaSuccess) return SHARQ_ECUDA;
      return cudaLaunchKernelEx(&lc, kfn, tm_sp, tm_dn, tm_w, p) == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
    }
  }
  using S = Stage<BN, FMT, false, AR, kExtra>;
  int64_t grid = tiles < env.num_sms ? tiles : env.num_sms;      // persistent: one CTA per SM
  if (debug_env().grid > 0) grid = debug_env().grid;
  if (env.plan_only) { fill_plan(env.plan_only, FUSED ? 4 : 0, BN, AR, 1, S::STAGES, tiles, grid, 1); return SHARQ_OK; }
  lc.gridDim = dim3((unsigned)grid);
  lc.dynamicSmemBytes = S::SMEM;
  if constexpr (FUSED) {
    static std::atomic<uint64_t> smem_set{0};
    auto kfn = sharq_linear_fused_kernel<BN, FMT, false, AR>;
    if (set_smem_once(smem_set, (const void*)kfn, S::SMEM, env.dev) != cudaSuccess) return SHARQ_ECUDA;
    return cudaLaunchKernelEx(&lc, kfn, tm_sp, tm_dn, tm_w, p, pp, norm) == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
  } else {
    if (p.path >= 3) {                                           // Table 5 combinations: second K-loop, fourth tensor map
      static std::atomic<uint64_t> smem_set{0};
      auto kfn = sharq_linear_combo_kernel<BN, FMT, AR>;
      if (set_smem_once(smem_set, (const void*)kfn, S::SMEM, env.dev) != cudaSuccess) return SHARQ_ECUDA;
      return cudaLaunchKernelEx(&lc, kfn, tm_sp, tm_dn, tm_w, tm_alt, p) == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
    }
    static std::atomic<uint64_t> smem_set{0};
    auto kfn = sharq_linear_kernel<BN, FMT, false, AR>;
    if (set_smem_once(smem_set, (const void*)kfn, S::SMEM, env.dev) != cudaSuccess) return SHARQ_ECUDA;
    return cudaLaunchKernelEx(&lc, kfn, tm_sp, tm_dn, tm_w, p) == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
  }
}

template <int BN, int FMT, int AR>
sharq_status launch_1cta(const LinearArgs& a, const KParams& p, const CUtensorMap& tm_sp,
                         const CUtensorMap& tm_dn, const CUtensorMap& tm_w, const CUtensorMap& tm_alt, int64_t tiles,
                         const LaunchEnv& env) {
  if constexpr (AR == 16) {                                // the fused decode launch exists for T <= 8 (8-row boxes) only
    if (env.fz) return launch_1cta_impl<BN, FMT, AR, true>(a, p, tm_sp, tm_dn, tm_w, tm_alt, tiles, env);
  }
  return launch_1cta_impl<BN, FMT, AR, false>(a, p, tm_sp, tm_dn, tm_w, tm_alt, tiles, env);
}

// grouped GEMM: persistent clusters of two CTAs on neighbouring n-tiles, activation operands multicast
template <int BN, int FMT, int MC>
sharq_status launch_mc_impl(const KParams& p, const CUtensorMap& tm_sp, const CUtensorMap& tm_dn,
                       const CUtensorMap& tm_w, int64_t tiles, const LaunchEnv& env) {
  using S = Stage<BN, FMT, false, 128, MC == 2 ? kStageBytes : 0>;
  auto kfn = sharq_linear_kernel<BN, FMT, false, 128, MC>;
  const int64_t clusters = tiles / 2 < env.num_sms / 2 ? tiles / 2 : env.num_sms / 2;
  if (env.plan_only) { fill_plan(env.plan_only, 2, BN, 128, 1, S::STAGES, tiles, 2 * clusters, 2); return SHARQ_OK; }
  static std::atomic<uint64_t> smem_set{0};
  if (set_smem_once(smem_set, (const void*)kfn, S::SMEM, env.dev) != cudaSuccess) return SHARQ_ECUDA;
  cudaLaunchConfig_t lc{};
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = debug_env().no_pdl ? 0 : 1;
  attr[1].id = cudaLaunchAttributeClusterDimension;
  attr[1].val.clusterDim.x = 2;
  attr[1].val.clusterDim.y = 1;
  attr[1].val.clusterDim.z = 1;
  lc.attrs = attr;
  lc.numAttrs = 2;
  lc.blockDim = dim3(MC == 2 ? kThreads + 128 : kThreads);
  lc.gridDim = dim3((unsigned)(2 * clusters));
  lc.dynamicSmemBytes = S::SMEM;
  lc.stream = env.st;
  return cudaLaunchKernelEx(&lc, kfn, tm_sp, tm_dn, tm_w, p) == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}

template <int BN, int FMT>
sharq_status launch_mc(const KParams& p, const CUtensorMap& tm_sp, const CUtensorMap& tm_dn,
                       const CUtensorMap& tm_w, int64_t tiles, const LaunchEnv& env) {
  if constexpr (BN == 128) {
    // tiles of at most four k-blocks are bound by their drain and stores: eight epilogue warps, three stages
    if (p.K <= 1024) return launch_mc_impl<128, FMT, 2>(p, tm_sp, tm_dn, tm_w, tiles, env);
  }
  return launch_mc_impl<BN, FMT, 1>(p, tm_sp, tm_dn, tm_w, tiles, env);
}

// scale-factor / metadata array as a 2-D tensor of 1024-byte rows (256 x u32), boxes of `box_rows` rows
bool make_map_rows1k(CUtensorMap* m, const void* base, uint64_t bytes, uint32_t box_rows) {
  EncodeTiledFn fn = encode_fn();
  if (!fn || bytes % 1024 != 0) return false;
  cuuint64_t dims[2] = {256, bytes / 1024};
  cuuint64_t strides[1] = {1024};
  cuuint32_t box[2] = {256, box_rows};
  cuuint32_t estr[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int FMT, int PBN, bool GROUPED = false>
sharq_status launch_pair(const LinearArgs& a, const KParams& p, const CUtensorMap& tm_sp, const CUtensorMap& tm_dn,
                         int64_t m_blocks, const LaunchEnv& env) {
  using P = PairStage<FMT, PBN>;
  constexpr int kSmem = GROUPED ? P::SMEM_GROUPED : P::SMEM;
  const int64_t n_tiles = (a.D + PBN - 1) / PBN;
  // grouped: the real number of pairs is only known on the device; an upper bound sizes the persistent grid
  const int64_t pair_tiles = (GROUPED ? (m_blocks + 1) / 2 + p.E : (m_blocks + 1) / 2) * n_tiles;
  int64_t clusters = pair_tiles < env.num_sms / 2 ? pair_tiles : env.num_sms / 2;
  if (debug_env().pair_clusters > 0 && debug_env().pair_clusters < clusters) clusters = debug_env().pair_clusters;
  if (env.plan_only) { fill_plan(env.plan_only, GROUPED ? 5 : 1, PBN, 128, 1, P::STAGES, pair_tiles, 2 * clusters, 2); return SHARQ_OK; }
  CUtensorMap tm_wp, tm_sfa_sp, tm_sfa_dn, tm_meta, tm_sfb_sp, tm_sfb_dn;
  const uint64_t act_rows = (uint64_t)m_blocks * 128, kk = (uint64_t)a.K;
  const uint32_t dn_rows = P::SF_DN_BYTES / 1024;
  const uint64_t dn_div = (FMT == SHARQ_NVFP4) ? 16 : 32;
  const uint64_t w_rows = (uint64_t)a.D * (uint64_t)(GROUPED ? p.E : 1);                // stacked experts
  const uint64_t w_rows_pad = (uint64_t)round_up((int64_t)w_rows, 128);   // the scale views are padded to whole 128-row atoms
  if (!make_map(&tm_wp, a.w_codes, w_rows, kk / 2, 128, P::HALF) ||
      !make_map_rows1k(&tm_sfa_sp, a.sp_sf, act_rows * kk / 32, 1) ||
      !make_map_rows1k(&tm_sfa_dn, a.dn_sf, act_rows * kk / dn_div, dn_rows) ||
      !make_map_rows1k(&tm_meta, a.sp_meta, act_rows * kk / 16, 2) ||
      !make_map_rows1k(&tm_sfb_sp, a.w_sf_sp, w_rows_pad * kk / 32, 1) ||
      !make_map_rows1k(&tm_sfb_dn, a.w_sf_dn, w_rows_pad * kk / dn_div, dn_rows))
    return SHARQ_ECUDA;
  auto kfn = sharq_linear_pair_kernel<FMT, PBN, GROUPED>;
  static std::atomic<uint64_t> smem_set{0};
  if (set_smem_once(smem_set, (const void*)kfn, kSmem, env.dev) != cudaSuccess) return SHARQ_ECUDA;
  cudaLaunchConfig_t lp{};
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = 2;
  at[0].val.clusterDim.y = 1;
  at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[1].val.programmaticStreamSerializationAllowed = debug_env().no_pdl ? 0 : 1;
  lp.blockDim = dim3(kThreads);
  lp.gridDim = dim3((unsigned)(2 * clusters));
  lp.dynamicSmemBytes = kSmem;
  lp.stream = env.st;
  lp.attrs = at;
  lp.numAttrs = 2;
  return cudaLaunchKernelEx(&lp, kfn, tm_sp, tm_dn, tm_wp, tm_sfa_sp, tm_sfa_dn, tm_meta, tm_sfb_sp, tm_sfb_dn, p) ==
                 cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}

// rows_total = rows the activation tensor maps cover (T; grouped: the capacity of the caller's padded buffers)
template <int BN, int FMT>
sharq_status launch_tiles(const LinearArgs& a, int64_t rows_total, int64_t m_blocks, int E, const int32_t* offsets,
                          const LaunchEnv& env) {
  const int num_sms = env.num_sms;
  CUtensorMap tm_sp, tm_dn, tm_w, tm_alt;
  const int64_t w_rows = (int64_t)(E > 0 ? E : 1) * a.D;
  const uint32_t a_rows = (E == 0 && m_blocks == 1 && rows_total < BM) ? (uint32_t)((rows_total + 7) / 8 * 8) : BM;
  // combinations: both operands are of one kind, the first in the sp_* (path 4) / dn_* (path 3) slots of the kernel
  const bool dd = a.path == 3, ss = a.path == 4;
  const void* first_dn = dd ? a.sp_codes : a.dn_codes;     // path 3: operand 0 arrives in the "sp" arguments of the ABI
  if (!env.plan_only &&
      (!make_map(&tm_sp, dd ? a.dn_codes : a.sp_codes, (uint64_t)rows_total, (uint64_t)a.K / (dd ? 2 : 4), dd ? 128 : 64, a_rows) ||
       !make_map(&tm_dn, ss ? a.sp_codes : first_dn, (uint64_t)rows_total, (uint64_t)a.K / (ss ? 4 : 2), ss ? 64 : 128, a_rows) ||
       !make_map(&tm_alt, a.dn_codes, (uint64_t)rows_total, (uint64_t)a.K / (ss ? 4 : 2), ss ? 64 : 128, a_rows) ||
       !make_map(&tm_w, a.w_codes, (uint64_t)w_rows, (uint64_t)a.K / 2, 128, BN < 256 ? BN : 256)))
    return SHARQ_ECUDA;
  const int64_t n_tiles = (a.D + BN - 1) / BN;               // the last n-tile may be ragged (D % 8 == 0): W rows beyond D
                                                             // are zero-filled by TMA, their columns never stored
  const int64_t tiles = m_blocks * n_tiles;                  // grouped: an upper bound (the kernel knows the real count)
  // path 3: kernel slots dn_sf = operand 0's scales (ABI: sp_sf), sf2 = operand 1's (ABI: dn_sf)
  // path 4: kernel slots sp_sf / sp_meta = operand 0, sf2 / meta2 = operand 1 (ABI: dn_sf / dn_meta)
  KParams p{(const uint8_t*)a.sp_sf, (const uint8_t*)a.sp_meta, (const uint8_t*)(dd ? a.sp_sf : a.dn_sf),
            (const uint8_t*)a.w_sf_sp, (const uint8_t*)a.w_sf_dn, a.row_scale, a.w_ts, (const uint16_t*)a.bias, a.Y, a.ldy,
            (int32_t)a.T, (int32_t)a.D, (int32_t)a.K, a.out_dtype, a.path, (int32_t)m_blocks,
            (int32_t)(E > 0 ? n_tiles : tiles), offsets, (int32_t)E, (const uint8_t*)a.dn_sf, (const uint8_t*)a.dn_meta,
            0, (int32_t)a_rows};
  const bool pair_worth = ((m_blocks + 1) / 2) * ((a.D + 255) / 256) >= num_sms / 4 || debug_env().force_pair;
  if (E == 0 && m_blocks >= 2 && BN == 128 && pair_worth && !debug_env().no_pair && a.path < 3) {
    // tile width by a cost model fitted on the box over the eight Llama / Qwen prefill shapes at T = 2048 ..
    // 8192 (us per round of 74 tiles): 256-wide 0.54 per k-block + 4.5 (one TMEM accumulator: drain and pipeline
    // refill exposed), 192-wide 0.50 per k-block + 1.5 (drain hidden by the second accumulator, but more
    // activation re-reads per output, which costs on long K)
    const int64_t clusters = num_sms / 2, m_pairs = (m_blocks + 1) / 2;
    const double kb = (double)(a.K / BK);
    const double cost192 = (double)((m_pairs * ((a.D + 191) / 192) + clusters - 1) / clusters) * (0.4975 * kb + 1.54);
    const double cost256 = (double)((m_pairs * ((a.D + 255) / 256) + clusters - 1) / clusters) * (0.5375 * kb + 4.5);
    int width = (a.D % 256 != 0 || cost192 < cost256) ? 192 : 256;
    if (debug_env().pair_bn > 0) width = (debug_env().pair_bn == 256 && a.D % 256 == 0) ? 256 : 192;
    // supertile height: the whole activation operand when it sits comfortably in L2 beside the streamed W tiles,
    // otherwise as many 256-row blocks as fit beside (the resident part of) W in ~72 MB of the 126 MB L2
    const double a_pair = 256.0 * (double)a.K * 0.90625, a_total = a_pair * (double)m_pairs;
    const double w_total = (double)a.D * (double)a.K * 0.59375;
    if (a_total > 48e6) {
      const double room = 72e6 - (w_total < 40e6 ? w_total : 40e6);
      int64_t gm = (int64_t)(room / a_pair);
      p.group_m = (int32_t)(gm < 1 ? 1 : gm > m_pairs ? m_pairs : gm);
    }
    if (debug_env().pair_gm > 0) p.group_m = debug_env().pair_gm;
    if (width == 256) return launch_pair<FMT, 256>(a, p, tm_sp, tm_dn, m_blocks, env);
    return launch_pair<FMT, 192>(a, p, tm_sp, tm_dn, m_blocks, env);
  }
  if constexpr (BN == 128) {
    // experts with (on average) well over 128 rows AND a long K: CTA-pair tiles, two row blocks of one expert x 192
    // columns per pair (half the weight bytes staged per CTA, M = 256 MMAs).  Short K-loops (BASELINE configs[4]:
    // K = 2048 / 768, 8 / 3 k-blocks per tile) are bound by the per-tile drain and store, not by the MMAs: measured
    // 134 / 114 us with pair tiles against 127 / 86 us with the 128-row multicast tiles below, so those stay there.
    if (E > 0 && rows_total / E >= 192 && a.K >= 4096 && !debug_env().no_pair)
      return launch_pair<FMT, 192, true>(a, p, tm_sp, tm_dn, m_blocks, env);
    // experts: n-tiles of one 128-row block are consecutive (decode_unit), so tiles 2j and 2j+1 share activations
    if (E > 0 && n_tiles % 2 == 0 && !debug_env().no_mc) return launch_mc<128, FMT>(p, tm_sp, tm_dn, tm_w, tiles, env);
  }
  if constexpr (BN == 192) {                               // launch_linear sends only grouped calls with an even n-tile count here
    return launch_mc<192, FMT>(p, tm_sp, tm_dn, tm_w, tiles, env);
  } else {
  if (a_rows <= 16) return launch_1cta<BN, FMT, 16>(a, p, tm_sp, tm_dn, tm_w, tm_alt, tiles, env);
  if (a_rows <= 64) return launch_1cta<BN, FMT, 64>(a, p, tm_sp, tm_dn, tm_w, tm_alt, tiles, env);
  return launch_1cta<BN, FMT, 128>(a, p, tm_sp, tm_dn, tm_w, tm_alt, tiles, env);
  }
}

}  // namespace

size_t hif4_linear_workspace_bytes(int64_t T, int64_t D, int64_t K);
sharq_status launch_linear_hif4(const LinearArgs& a, void* workspace, size_t workspace_bytes, int num_sms,
                                cudaStream_t st);

size_t linear_workspace_bytes(const sharq_config* cfg, int64_t T, int64_t D, int64_t K, int32_t) {
  return cfg->fmt == SHARQ_HIF4 ? hif4_linear_workspace_bytes(T, D, K) : 0;   // bf16 copies of A and W
}

// E > 0: grouped; `offsets` is the DEVICE int32[E + 1] array, a.T the row capacity of the padded activation buffers.
// plan_only != nullptr: fill it with the launch configuration this call would use and launch nothing.
sharq_status launch_linear(const sharq_config* cfg, const LinearArgs& a, int32_t E, const int32_t* offsets,
                           void* workspace, size_t workspace_bytes, int num_sms, int dev, cudaStream_t st,
                           LinearPlan* plan_only, const FusedArgs* fz) {
  if (cfg->fmt == SHARQ_HIF4) {                           // no FP4-rate tensor path: exact bf16 emulation
    if (E > 0) return SHARQ_EINVAL;
    if (plan_only) {
      const int bn = a.D % 256 == 0 ? 256 : 128;
      const int64_t tiles = ((a.T + 127) / 128) * (a.D / bn);
      fill_plan(plan_only, 3, bn, 128, 1, bn == 256 ? 4 : 6, tiles, tiles < num_sms ? tiles : num_sms, 1);
      return SHARQ_OK;
    }
    return launch_linear_hif4(a, workspace, workspace_bytes, num_sms, st);
  }
  if (a.K > (int64_t)1 << 24 || a.D > (int64_t)1 << 24 || a.T > (int64_t)1 << 30) return SHARQ_ESHAPE;
  const LaunchEnv env{num_sms, dev, st, plan_only, fz};
  int64_t rows_total = a.T, m_blocks = (a.T + BM - 1) / BM;
  if (E > 0) {
    if (E > kMaxExperts) return SHARQ_ESHAPE;
    m_blocks = a.T / BM;                                  // whole 128-row blocks of the caller's buffers
    rows_total = m_blocks * BM;
    if (m_blocks == 0) return SHARQ_OK;
  }
  if (m_blocks * ((a.D + 127) / 128) > (int64_t)1 << 30) return SHARQ_ESHAPE;
  if (E > 0 && a.D % 128 != 0) return SHARQ_ESHAPE;       // stacked expert weights: whole 128-row scale atoms per expert
  // T <= 128 (one m-block): 128 x 256 tiles halve the per-column cost of the scale-factor copies and of the M = 128 MMA
  // (the decode launches are bound by tensor-pipe issue per k-block, not by HBM)
  // ... and only pays when the 128-wide tiles would need a second round on the SMs (measured: with fewer
  // tiles than SMs the narrower tiles + deeper K-split win)
  if (E == 0 && a.path < 3 && a.T <= debug_env().wide_t && a.D % 256 == 0 && a.D / 128 > num_sms && !debug_env().no_wide) {
    if (cfg->fmt == SHARQ_NVFP4) return launch_tiles<256, SHARQ_NVFP4>(a, rows_total, m_blocks, E, offsets, env);
    return launch_tiles<256, SHARQ_MXFP4>(a, rows_total, m_blocks, E, offsets, env);
  }
  // experts with a medium K-loop (more than four k-blocks per tile, too short for the grouped pair tiles): 128 x 192
  // tiles in multicast clusters.  Those launches are bound by the bytes each SM takes in per k-block (~85 GB/s per SM:
  // operands of a 128 x 128 tile 48 KB, of a 128 x 192 tile 59 KB for 1.5 x the flop)
  const bool pair_grouped = E > 0 && rows_total / E >= 192 && a.K >= 4096 && !debug_env().no_pair;
  if (E > 0 && a.D % 384 == 0 && a.K > 1024 && !pair_grouped && !debug_env().no_mc) {
    if (cfg->fmt == SHARQ_NVFP4) return launch_tiles<192, SHARQ_NVFP4>(a, rows_total, m_blocks, E, offsets, env);
    return launch_tiles<192, SHARQ_MXFP4>(a, rows_total, m_blocks, E, offsets, env);
  }
  if (cfg->fmt == SHARQ_NVFP4) return launch_tiles<128, SHARQ_NVFP4>(a, rows_total, m_blocks, E, offsets, env);
  return launch_tiles<128, SHARQ_MXFP4>(a, rows_total, m_blocks, E, offsets, env);
}

#if defined(SHARQ_EXPERIMENTS) && defined(SHARQ_DEBUG_TS)
extern "C" int sharq_debug_read_ts(long long* host_out) {
  return (int)cudaMemcpyFromSymbol(host_out, g_dbg_ts, sizeof(long long) * 1024 * 16);
}
#endif
}  // namespace sharq
