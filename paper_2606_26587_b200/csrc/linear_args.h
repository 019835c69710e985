// Host-side argument bundle of sharq_linear / sharq_linear_grouped, shared by api.cu, linear.cu and linear_hif4.cu.
#pragma once
#include <stdint.h>

namespace sharq {

struct LinearArgs {
  int64_t T, D, K;              // T = rows (grouped: row capacity of the padded activation buffers)
  const void *sp_codes, *sp_sf, *sp_meta, *dn_codes, *dn_sf;   // paths 3 / 4: operand 0 (sp_*) and operand 1 (dn_*)
  const void* dn_meta;                                          // path 4 only: metadata of the second sparse operand
  const float* row_scale;
  const void *w_codes, *w_sf_sp, *w_sf_dn;
  const float* w_ts;
  const void* bias;
  void* Y; int64_t ldy; int out_dtype; int path;
};

// sharq_prepare_linear (N2): the in-kernel prepare of the fused decode launch; nullptr = plain sharq_linear
struct PrepParams;
struct FusedArgs {
  const PrepParams* pp;
  int32_t norm;        // SHARQ_NORM_NONE or SHARQ_NORM_RMS
  int32_t warps;       // prepare warps per CTA = ceil(K / 1024)
};

// what a sharq_linear call launches (sharq_linear_plan): kind 0 = 128-row tiles, one CTA per tile (persistent, or a
// split-K cluster of `splits` CTAs per tile); 1 = CTA-pair tiles (256 rows x bn); 2 = grouped GEMM, multicast
// clusters of two CTAs; 3 = HiF4 bf16 emulation
struct LinearPlan {
  int32_t kind, bn, act_rows, splits, stages, cluster;
  int64_t tiles, grid;
};

}  // namespace sharq
