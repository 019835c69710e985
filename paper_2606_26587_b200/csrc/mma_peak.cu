// sharq_mma_peak_launch: tensor-pipe issue-rate probe ("P_dn, P_sp = measured on the box by
// a TMEM-resident MMA issue loop").  One CTA pair per two SMs issues `iters` k-blocks (256 logical k) of the
// SAME instruction sequence sharq_linear_pair_kernel issues per k-block -- 2 x tcgen05.mma.sp + 4 x dense
// tcgen05.mma, M = 256, N = 256, optionally with the 19 tcgen05.cp of scale factors / metadata -- on whatever
// bytes are in shared memory, with no loads and no epilogue.  bench.py times it with CUDA events; the
// result is the ceiling of the GEMM's main loop on this GPU at the clocks of the moment.
#include <cuda_runtime.h>

#include "../../include/sharq_diag.h"
#include "common.cuh"
#include "tc_ptx.cuh"

namespace sharq {
namespace {

__device__ __forceinline__ uint32_t probe_hash(uint32_t x) {           // a 32-bit mixer (operand bits of the probe)
  x ^= x >> 16; x *= 0x7FEB352Du; x ^= x >> 15; x *= 0x846CA68Bu; x ^= x >> 16;
  return x;
}

// mode bits: 1 = dense MMAs, 2 = sparse MMAs, 4 = scale-factor / metadata copies, 8 = pseudo-random operand bits
// (uniform FP4 codes, finite scale bytes, valid metadata nibbles) instead of the constant 0x22 bytes: the GPU is
// power capped, and a tensor pipe fed constants switches far fewer bits than one fed data
__global__ void __launch_bounds__(128, 1) mma_peak_kernel(int iters, int mode) {
  extern __shared__ uint8_t raw[];
  const uint32_t base = (smem_u32(raw) + 1023u) & ~1023u;
  __shared__ uint64_t bar;
  __shared__ uint32_t tptr;
  const uint32_t bar_addr = smem_u32(&bar);
  if (threadIdx.x == 0) {
    tc::mbar_init(bar_addr, 1);
    tc::fence_mbar_init();
  }
  for (int i = threadIdx.x; i < 200 * 1024 / 4; i += 128) {
    uint32_t v = 0x22222222u;
    if (mode & 8) {
      const uint32_t addr = smem_u32(raw) + 4u * (uint32_t)i;
      const uint32_t off = addr >= base ? (addr - base) % 49152u : 0u;      // offset inside the 48 KB stage
      v = probe_hash((uint32_t)i * 2654435761u + blockIdx.x * 97u + 1u);
      if (off >= 43008u) {
        v = (v & 0x1F1F1F1Fu) | 0x30303030u;                    // UE4M3 scales in [2^-1, 2^2): finite, varied
      } else if (off >= 40960u) {                               // metadata: one of the six valid nibbles per chunk
        uint32_t m = 0, h = v;
#pragma unroll
        for (int q = 0; q < 8; ++q) { m |= ((0xED9C84u >> (4 * (h % 6u))) & 0xFu) << (4 * q); h = h / 6u + (h << 7); }
        v = m;
      }
    }
    reinterpret_cast<uint32_t*>(raw)[i] = v;
  }
  tc::fence_proxy_async();
  if (threadIdx.x < 32) tc::tmem_alloc_pair<512>(smem_u32(&tptr));
  tc::tc_fence_before();
  __syncthreads();
  tc::cluster_sync_all();
  tc::tc_fence_after();
  const uint32_t tb = tptr;
  if (threadIdx.x < 32 && tc::cluster_ctarank() == 0) {
    const bool lead = tc::elect_one() != 0;
    const uint32_t id_dn = tc::idesc_fp4(256, 256, false, false, 0, 0), id_sp = tc::idesc_fp4(256, 256, true, false, 0, 0);
    for (int it = 0; it < iters; ++it) {
      const uint32_t st = base + (it & 3) * 49152;
      if (mode & 4) {
        if (mode & 2) {
          if (lead) tc::tc_cp_meta_pair(tb + 256, tc::smem_desc(st + 40960, 128, 0));
#pragma unroll
          for (int a = 0; a < 6; ++a)
            if (lead) tc::tc_cp_sf_pair(tb + 260 + 4 * a, tc::smem_desc(st + 43008 + 512 * a, 128, 0));
        }
        if (mode & 1) {
#pragma unroll
          for (int a = 0; a < 12; ++a)
            if (lead) tc::tc_cp_sf_pair(tb + 300 + 4 * a, tc::smem_desc(st + 43008 + 512 * (a & 7), 128, 0));
        }
      }
      if (mode & 2) {
#pragma unroll
        for (int j = 0; j < 2; ++j)
          if (lead) tc::mma_sparse_pair(tb, tc::smem_desc(st + 32768 + 32 * j, 512, 4), tc::smem_desc(st + 16384 + 64 * j, 1024, 2),
                                        id_sp, tb + 260 + 4 * j, tb + 268 + 8 * j, tb + 256 + 2 * j, 1);
      }
      if (mode & 1) {
#pragma unroll
        for (int j = 0; j < 4; ++j)
          if (lead) tc::mma_dense_pair<true>(tb, tc::smem_desc(st + 32 * j, 1024, 2), tc::smem_desc(st + 16384 + 32 * j, 1024, 2),
                                             id_dn, tb + 300 + 4 * j, tb + 316 + 8 * j, 1);
      }
    }
    if (lead) tc::tc_commit_pair(bar_addr, 1);
    tc::mbar_wait(bar_addr, 0);
  }
  __syncthreads();
  tc::cluster_sync_all();
  if (threadIdx.x < 32) tc::tmem_dealloc_pair<512>(tb);
}

}  // namespace
}  // namespace sharq

extern "C" sharq_status sharq_mma_peak_launch(int32_t mode, int32_t iters, void* stream) {
  using namespace sharq;
  if (mode < 1 || mode > 15 || (mode & 3) == 0 || iters <= 0) return SHARQ_EINVAL;
  int dev = 0, major = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return SHARQ_ECUDA;
  cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (major != 10) return SHARQ_EARCH;
  const int smem = 200 * 1024 + 2048;
  if (cudaFuncSetAttribute(mma_peak_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess)
    return SHARQ_ECUDA;
  cudaLaunchConfig_t lc{};
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  lc.gridDim = dim3((unsigned)(sms / 2 * 2));
  lc.blockDim = dim3(128);
  lc.dynamicSmemBytes = smem;
  lc.stream = (cudaStream_t)stream;
  lc.attrs = at;
  lc.numAttrs = 1;
  return cudaLaunchKernelEx(&lc, mma_peak_kernel, (int)iters, (int)mode) == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}
