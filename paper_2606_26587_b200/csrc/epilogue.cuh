// Shared by the GEMM kernels of linear.cu and linear_hif4.cu: the epilogue through shared memory and the tile order of
// the CTA-pair kernels.  P = the kernel's parameter struct (fields bias, out_fp32, D, Y, ldy).
#pragma once
#include "common.cuh"
#include "tc_ptx.cuh"

namespace sharq {

constexpr int kStageBytes = 4 * 4096;      // epilogue staging: 4 KB for each of the four epilogue warps

// ---- epilogue through shared memory (persistent tiles and CTA pairs) ------------------------------------------
// tcgen05.ld hands every thread 32 consecutive columns of ITS row, so direct stores are 32 rows x 16 bytes per warp
// instruction: 32 half-filled sectors, and the LSU becomes the bound of short-K tiles (MoE experts: the tile's stores
// cost 31 % of the down projection).  Instead each epilogue warp stages 128 bytes per row (64 bf16 or 32 fp32 columns)
// of its 32 rows in its own 4 KB of shared memory (16-byte chunks XOR-swizzled by the row, conflict free both ways)
// and writes them back transposed: one warp instruction = 4 rows x one full 128-byte line.

__device__ __forceinline__ uint32_t stg_addr(uint32_t base, int r, int ch) {
  return base + (uint32_t)r * 128u + ((uint32_t)(ch ^ (r & 7)) << 4);
}

// y = acc * scale (+ bias) for the 32 columns col0 .. col0 + 31 of this thread's row, into the staging row `lane`;
// slot = which half of the 128 staged bytes a bf16 chunk takes (fp32: the whole row)
template <class P>
__device__ __forceinline__ void epilogue_stage32(const P& p, uint32_t stg, int lane, int col0, int slot, float scale,
                                                 const uint32_t (&v)[32]) {
  float f[32];
#pragma unroll
  for (int i = 0; i < 32; ++i) f[i] = __fmul_rn(__uint_as_float(v[i]), scale);
  if (p.bias) {
    const int ncols = p.D - col0;                     // < 32 only on a ragged last n-tile
    const uint16_t* b = p.bias + col0;
#pragma unroll
    for (int i = 0; i < 32; ++i)
      if (i < ncols) f[i] = __fadd_rn(f[i], __uint_as_float((uint32_t)b[i] << 16));
  }
  if (p.out_fp32) {
#pragma unroll
    for (int j = 0; j < 8; ++j) tc::st_shared_v4(stg_addr(stg, lane, j), f[4 * j], f[4 * j + 1], f[4 * j + 2], f[4 * j + 3]);
  } else {
#pragma unroll
    for (int j = 0; j < 4; ++j)
      tc::st_shared_v4(stg_addr(stg, lane, 4 * slot + j),
                       __uint_as_float(pack_bf16x2_rn(f[8 * j], f[8 * j + 1])), __uint_as_float(pack_bf16x2_rn(f[8 * j + 2], f[8 * j + 3])),
                       __uint_as_float(pack_bf16x2_rn(f[8 * j + 4], f[8 * j + 5])), __uint_as_float(pack_bf16x2_rn(f[8 * j + 6], f[8 * j + 7])));
  }
}

// the staged 32 rows x 128 bytes -> Y: rows row0 .. row0 + rows_ok - 1, columns from colbase, D-guarded per 16 bytes
template <class P>
__device__ __forceinline__ void epilogue_flush(const P& p, uint32_t stg, int lane, int64_t row0, int rows_ok, int colbase,
                                               int col_end) {
  const int ch = lane & 7;
  const int col = colbase + ch * (p.out_fp32 ? 4 : 8);
  uint8_t* ybase = static_cast<uint8_t*>(p.Y) + (size_t)col * (p.out_fp32 ? 4 : 2);
  const size_t pitch = (size_t)p.ldy * (p.out_fp32 ? 4 : 2);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int rr = 4 * i + (lane >> 3);
    if (rr < rows_ok && col < col_end) {
      const float4 t = tc::ld_shared_v4(stg_addr(stg, rr, ch));
      *reinterpret_cast<float4*>(ybase + (size_t)(row0 + rr) * pitch) = t;
    }
  }
}

// all BN columns of one accumulator stage of this warp's 32 rows.  PIPE: the tensor-memory load of chunk c + 1 is
// issued before chunk c is scaled, staged and stored (two register buffers, two chunks per loop iteration), so the load
// latency of every chunk but the first runs under the previous chunk's work.  (A FULLY unrolled version cost the decode
// launches, whose CTAs drain one or two tiles in their life, ~1 us each in cold instruction fetches.)
template <int BN, bool PIPE = true, class P>
__device__ __forceinline__ void epilogue_tile(const P& p, uint32_t taddr, uint32_t stg, int lane, int64_t row0, int rows_ok,
                                              int n0, float scale) {
  constexpr int NC = BN / 32;
  auto finish = [&](int c, const uint32_t (&v)[32]) {
    const bool second = !p.out_fp32 && (c & 1);
    epilogue_stage32(p, stg, lane, n0 + c * 32, second ? 1 : 0, scale, v);
    if (p.out_fp32 || second || c == NC - 1) {        // (a tile of an odd number of 32-column chunks: half a staged row)
      __syncwarp();
      epilogue_flush(p, stg, lane, row0, rows_ok, n0 + (second ? c - 1 : c) * 32, min(p.D, n0 + (c + 1) * 32));
      __syncwarp();
    }
  };
  if constexpr (PIPE) {
    uint32_t v0[32], v1[32];
    tc::tmem_ld32(taddr, v0);
#pragma unroll 1
    for (int c = 0; c < NC; c += 2) {                 // two chunks per iteration: compact code, two register buffers
      tc::tmem_ld_wait(v0);                           // chunk c has arrived (tcgen05.wait::ld covers every earlier load)
      if (c + 1 < NC) tc::tmem_ld32(taddr + (c + 1) * 32, v1);
      finish(c, v0);
      if (c + 1 < NC) {
        tc::tmem_ld_wait(v1);
        if (c + 2 < NC) tc::tmem_ld32(taddr + (c + 2) * 32, v0);
        finish(c + 1, v1);
      }
    }
  } else {
#pragma unroll 1
    for (int c = 0; c < NC; ++c) {
      uint32_t v[32];
      tc::tmem_ld32(taddr + c * 32, v);
      tc::tmem_ld_wait();
      finish(c, v);
    }
  }
}

// Tile order of the pair kernel.  Tiles run m-fastest inside a SUPERTILE of `gm` 256-row blocks x all n-tiles: the
// concurrently running clusters then touch gm activation blocks (which stay in L2 for the whole supertile, read from
// DRAM once) and one or two W tiles at a time.  gm = all row blocks reproduces the plain m-fastest order (right when
// the whole activation operand fits in L2); with a long K and many tokens (down projection at T = 8192: 106 MB of
// activation operands) the plain order cycled the whole operand through L2 once per two n-tiles: 782 MB of DRAM
// reads for 137 MB of operands (profiles/linear_pair_r2_ncu_full.md).
__device__ __forceinline__ void pair_tile(int tile, int m_pairs, int n_tiles, int gm, int& m_pair, int& n_blk) {
  const int per_group = gm * n_tiles;
  const int g = tile / per_group;
  const int g0 = g * gm;
  const int rows = min(gm, m_pairs - g0);              // the last supertile may be shorter
  const int within = tile - g * per_group;
  m_pair = g0 + within % rows;
  n_blk = within / rows;
}


}  // namespace sharq
