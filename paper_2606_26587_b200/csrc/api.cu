// C ABI of libsharq.so (include/sharq.h): argument validation, size queries, dispatch.
// All compute is in prepare.cu / linear.cu; there is no CPU fallback anywhere.
#include <cuda_runtime.h>
#include <stdio.h>

#include "common.cuh"
#include "linear_args.h"
#include "prepare_device.cuh"

namespace sharq {
cudaError_t launch_prepare(const sharq_config* cfg, const void* x, int64_t T, int64_t K, int64_t ldx,
                           const void* gamma, const void* beta, const float* x_ts, void* sp_codes, void* sp_sf,
                           void* sp_meta, void* dn_codes, void* dn_sf, float* row_scale, int num_sms,
                           cudaStream_t st, const void* residual, int64_t ldr, void* sum_out, int64_t ldo,
                           int combo, void* dn_meta);
cudaError_t launch_quantize_weight(const sharq_config* cfg, const void* W, int64_t D, int64_t K, int64_t ldw,
                                   void* codes, void* sf_sp, void* sf_dn, float* ts, void* workspace,
                                   cudaStream_t st);
sharq_status launch_linear(const sharq_config* cfg, const LinearArgs& a, int32_t E, const int32_t* offsets,
                           void* workspace, size_t workspace_bytes, int num_sms, int dev, cudaStream_t st,
                           LinearPlan* plan_only, const FusedArgs* fz = nullptr);
PrepParams make_prep_params(const sharq_config* cfg, const void* x, int64_t T, int64_t K, int64_t ldx, const void* gamma,
                            const void* beta, const float* x_ts, void* sp_codes, void* sp_sf, void* sp_meta,
                            void* dn_codes, void* dn_sf, float* row_scale);
cudaError_t launch_untile(const void* tiled, int64_t R, int64_t C, void* canonical, int meta, cudaStream_t st);
size_t linear_workspace_bytes(const sharq_config* cfg, int64_t T, int64_t D, int64_t K, int32_t E);
}  // namespace sharq

using namespace sharq;

namespace {

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

sharq_status check_cfg(const sharq_config* cfg) {
  if (!cfg) return SHARQ_EINVAL;
  if (cfg->fmt < 0 || cfg->fmt > 2 || cfg->mask < 0 || cfg->mask > 1 || cfg->norm < 0 || cfg->norm > 2 ||
      cfg->layout < 0 || cfg->layout > 1)
    return SHARQ_EINVAL;
  // HiF4 uses the standard 2:4; for NVFP4 / MXFP4 the element-wise 2:4 is an encoding the oracle can check
  // (sharq_prepare, canonical layout) but not one the block-scaled FP4 sparse MMA takes (check_linear refuses it)
  if (cfg->fmt == SHARQ_HIF4 && cfg->mask != SHARQ_MASK_24) return SHARQ_EINVAL;
  if (cfg->mask == SHARQ_MASK_24 && cfg->layout != SHARQ_LAYOUT_CANONICAL) return SHARQ_EINVAL;
  return SHARQ_OK;
}

struct DeviceInfo { int ok; int sms; int major; int dev; };
sharq_status device_info(DeviceInfo* out) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return SHARQ_ECUDA;
  int major = 0, sms = 0;
  if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return SHARQ_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return SHARQ_ECUDA;
  if (major != 10) return SHARQ_EARCH;
  out->ok = 1; out->sms = sms; out->major = major; out->dev = dev;
  return SHARQ_OK;
}

int64_t sf_cols(int fmt, bool dense_group, int64_t K) {
  if (fmt == SHARQ_HIF4) return K / 64 * 4;                       // uint32 words, in bytes
  if (fmt == SHARQ_NVFP4 && dense_group) return K / 16;
  return K / 32;
}
size_t sf_bytes(const sharq_config* cfg, int64_t rows, int64_t cols_bytes) {
  return (size_t)((cfg->layout == SHARQ_LAYOUT_TILED) ? round_up(rows, 128) : rows) * (size_t)cols_bytes;
}

}  // namespace

extern "C" {

const char* sharq_version(void) { return "sharq-b200 0.1 sm_100a"; }

sharq_status sharq_weight_sizes(const sharq_config* cfg, int64_t D, int64_t K, size_t* codes, size_t* sf_sparse_view,
                                size_t* sf_dense_view, size_t* workspace) {
  sharq_status s = check_cfg(cfg);
  if (s != SHARQ_OK) return s;
  if (D < 0 || K <= 0 || K % 256 != 0) return SHARQ_ESHAPE;
  if (codes) *codes = (size_t)D * (size_t)(K / 2);
  if (sf_sparse_view) *sf_sparse_view = sf_bytes(cfg, D, sf_cols(cfg->fmt, false, K));
  if (sf_dense_view)                                       // HiF4: the exact bf16 dequantisation [D, K] (the GEMM-side view)
    *sf_dense_view = cfg->fmt == SHARQ_HIF4 ? (size_t)D * (size_t)K * 2 : sf_bytes(cfg, D, sf_cols(cfg->fmt, true, K));
  if (workspace) *workspace = 256;
  return SHARQ_OK;
}

sharq_status sharq_act_sizes(const sharq_config* cfg, int64_t T, int64_t K, size_t* sp_codes, size_t* sp_sf,
                             size_t* sp_meta, size_t* dn_codes, size_t* dn_sf, size_t* row_scale) {
  sharq_status s = check_cfg(cfg);
  if (s != SHARQ_OK) return s;
  if (T < 0 || K <= 0 || K % 256 != 0) return SHARQ_ESHAPE;
  if (sp_codes) *sp_codes = (size_t)T * (size_t)(K / 4);
  if (sp_sf) *sp_sf = sf_bytes(cfg, T, sf_cols(cfg->fmt, false, K));
  if (sp_meta) *sp_meta = sf_bytes(cfg, T, cfg->mask == SHARQ_MASK_24 ? K / 8 : K / 16);
  if (dn_codes) *dn_codes = (size_t)T * (size_t)(K / 2);
  if (dn_sf) *dn_sf = sf_bytes(cfg, T, sf_cols(cfg->fmt, true, K));
  if (row_scale) *row_scale = (size_t)T * sizeof(float);
  return SHARQ_OK;
}

sharq_status sharq_linear_workspace(const sharq_config* cfg, int64_t T, int64_t D, int64_t K, int32_t E,
                                    size_t* workspace) {
  sharq_status s = check_cfg(cfg);
  if (s != SHARQ_OK) return s;
  if (T < 0 || D <= 0 || D % 8 != 0 || K <= 0 || K % 256 != 0 || E < 0) return SHARQ_ESHAPE;
  if ((cfg->fmt == SHARQ_HIF4 || E > 0) && D % 128 != 0) return SHARQ_ESHAPE;
  if (cfg->fmt != SHARQ_HIF4 && cfg->mask != SHARQ_MASK_PAIR48) return SHARQ_ESHAPE;
  if (workspace) *workspace = linear_workspace_bytes(cfg, T, D, K, E);
  return SHARQ_OK;
}

sharq_status sharq_quantize_weight(const sharq_config* cfg, const void* W, int64_t D, int64_t K, int64_t ldw,
                                   void* codes, void* sf_sparse_view, void* sf_dense_view, float* tensor_scale,
                                   void* workspace, size_t workspace_bytes, void* stream) {
  sharq_status s = check_cfg(cfg);
  if (s != SHARQ_OK) return s;
  if (D < 0 || K <= 0 || K % 256 != 0 || ldw < K || ldw % 8 != 0) return SHARQ_ESHAPE;
  if (!W || !codes || !sf_sparse_view || !sf_dense_view || !tensor_scale || !workspace) return SHARQ_EINVAL;
  if (!aligned16(W) || !aligned16(codes) || !aligned16(sf_sparse_view) || !aligned16(sf_dense_view) ||
      !aligned16(workspace))
    return SHARQ_EINVAL;
  if (workspace_bytes < 256) return SHARQ_EWORKSPACE;
  DeviceInfo di{};
  if ((s = device_info(&di)) != SHARQ_OK) return s;
  if (D == 0) return SHARQ_OK;
  cudaError_t e = launch_quantize_weight(cfg, W, D, K, ldw, codes, sf_sparse_view, sf_dense_view, tensor_scale,
                                         workspace, (cudaStream_t)stream);
  return e == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}

sharq_status sharq_prepare(const sharq_config* cfg, const void* x, int64_t T, int64_t K, int64_t ldx,
                           const void* gamma, const void* beta, const float* x_tensor_scale, void* sp_codes,
                           void* sp_sf, void* sp_meta, void* dn_codes, void* dn_sf, float* row_scale, void* stream) {
  sharq_status s = check_cfg(cfg);
  if (s != SHARQ_OK) return s;
  if (T < 0 || K <= 0 || K % 256 != 0 || ldx < K || ldx % 8 != 0) return SHARQ_ESHAPE;
  if (T == 0) return SHARQ_OK;
  if (!x || !sp_codes || !sp_sf || !sp_meta || !dn_codes || !dn_sf || !row_scale) return SHARQ_EINVAL;
  if (cfg->norm != SHARQ_NORM_NONE && !gamma) return SHARQ_EINVAL;
  if (!aligned16(x) || !aligned16(sp_codes) || !aligned16(sp_sf) || !aligned16(sp_meta) || !aligned16(dn_codes) ||
      !aligned16(dn_sf) || (gamma && !aligned16(gamma)) || (beta && !aligned16(beta)))
    return SHARQ_EINVAL;
  if (K > 100 * 1024) return SHARQ_ESHAPE;   // one row must fit in shared memory
  DeviceInfo di{};
  if ((s = device_info(&di)) != SHARQ_OK) return s;
  cudaError_t e = launch_prepare(cfg, x, T, K, ldx, gamma, beta, x_tensor_scale, sp_codes, sp_sf, sp_meta, dn_codes,
                                 dn_sf, row_scale, di.sms, (cudaStream_t)stream, nullptr, 0, nullptr, 0, 0, nullptr);
  return e == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}

sharq_status sharq_prepare_add(const sharq_config* cfg, const void* x, const void* residual, int64_t T, int64_t K,
                               int64_t ldx, int64_t ldr, void* sum_out, int64_t ldo, const void* gamma,
                               const void* beta, const float* x_tensor_scale, void* sp_codes, void* sp_sf,
                               void* sp_meta, void* dn_codes, void* dn_sf, float* row_scale, void* stream) {
  sharq_status s = check_cfg(cfg);
  if (s != SHARQ_OK) return s;
  if (T < 0 || K <= 0 || K % 256 != 0 || K > 32768) return SHARQ_ESHAPE;
  if (cfg->fmt == SHARQ_NVFP4 && cfg->norm == SHARQ_NORM_LAYER && K > 25600) return SHARQ_ESHAPE;   // one row per CTA no longer fits
  if (cfg->fmt != SHARQ_HIF4 && cfg->mask != SHARQ_MASK_PAIR48) return SHARQ_EINVAL;   // the fused add has no 2:4 E2M1 variant
  if (ldx < K || ldr < K || ldo < K || ldx % 16 != 0 || ldr % 16 != 0 || ldo % 16 != 0) return SHARQ_ESHAPE;
  if (T == 0) return SHARQ_OK;
  if (!x || !residual || !sum_out || !sp_codes || !sp_sf || !sp_meta || !dn_codes || !dn_sf || !row_scale) return SHARQ_EINVAL;
  if (cfg->norm != SHARQ_NORM_NONE && !gamma) return SHARQ_EINVAL;
  auto aligned32 = [](const void* q) { return ((uintptr_t)q & 31u) == 0; };
  if (!aligned32(x) || !aligned32(residual) || !aligned32(sum_out)) return SHARQ_EINVAL;
  if (!aligned16(sp_codes) || !aligned16(sp_sf) || !aligned16(sp_meta) || !aligned16(dn_codes) || !aligned16(dn_sf) ||
      (gamma && !aligned16(gamma)) || (beta && !aligned16(beta)))
    return SHARQ_EINVAL;
  if (sum_out == x) return SHARQ_EINVAL;   // x is re-read by the software pipeline one row ahead; residual may alias sum_out
  DeviceInfo di{};
  if ((s = device_info(&di)) != SHARQ_OK) return s;
  cudaError_t e = launch_prepare(cfg, x, T, K, ldx, gamma, beta, x_tensor_scale, sp_codes, sp_sf, sp_meta, dn_codes,
                                 dn_sf, row_scale, di.sms, (cudaStream_t)stream, residual, ldr, sum_out, ldo, 0, nullptr);
  return e == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}

// sharq_prepare with h = bf16(silu(gate) * up) computed on the fly (the row kernel's fused-operand path with no
// sum_out: the activation never goes to HBM)
sharq_status sharq_prepare_swiglu(const sharq_config* cfg, const void* gate, const void* up, int64_t T, int64_t K,
                                  int64_t ldg, int64_t ldu, const void* gamma, const void* beta,
                                  const float* x_tensor_scale, void* sp_codes, void* sp_sf, void* sp_meta,
                                  void* dn_codes, void* dn_sf, float* row_scale, void* stream) {
  sharq_status s = check_cfg(cfg);
  if (s != SHARQ_OK) return s;
  if (T < 0 || K <= 0 || K % 256 != 0 || K > 32768) return SHARQ_ESHAPE;
  if (cfg->norm != SHARQ_NORM_NONE) return SHARQ_EINVAL;   // the down projection's input is not normalised
  if (cfg->fmt != SHARQ_HIF4 && cfg->mask != SHARQ_MASK_PAIR48) return SHARQ_EINVAL;
  if (ldg < K || ldu < K || ldg % 16 != 0 || ldu % 16 != 0) return SHARQ_ESHAPE;
  if (T == 0) return SHARQ_OK;
  if (!gate || !up || !sp_codes || !sp_sf || !sp_meta || !dn_codes || !dn_sf || !row_scale) return SHARQ_EINVAL;
  if (cfg->norm != SHARQ_NORM_NONE && !gamma) return SHARQ_EINVAL;
  if (((uintptr_t)gate & 31u) || ((uintptr_t)up & 31u)) return SHARQ_EINVAL;
  if (!aligned16(sp_codes) || !aligned16(sp_sf) || !aligned16(sp_meta) || !aligned16(dn_codes) || !aligned16(dn_sf) ||
      (gamma && !aligned16(gamma)) || (beta && !aligned16(beta)))
    return SHARQ_EINVAL;
  DeviceInfo di{};
  if ((s = device_info(&di)) != SHARQ_OK) return s;
  cudaError_t e = launch_prepare(cfg, gate, T, K, ldg, gamma, beta, x_tensor_scale, sp_codes, sp_sf, sp_meta, dn_codes,
                                 dn_sf, row_scale, di.sms, (cudaStream_t)stream, up, ldu, nullptr, 0, 0, nullptr);
  return e == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}

static sharq_status check_linear(const sharq_config* cfg, int64_t D, int64_t K, const void* const* ptrs, int n,
                                 int64_t ldy, int32_t out_dtype, int32_t path) {
  sharq_status s = check_cfg(cfg);
  if (s != SHARQ_OK) return s;
  if (cfg->fmt != SHARQ_HIF4 && cfg->mask != SHARQ_MASK_PAIR48) return SHARQ_ESHAPE;   // no element-wise 2:4 FP4 MMA
  if (cfg->layout != SHARQ_LAYOUT_TILED && cfg->fmt != SHARQ_HIF4) return SHARQ_EINVAL;
  if (D <= 0 || D % 8 != 0 || K <= 0 || K % 256 != 0 || ldy < D || ldy % 8 != 0) return SHARQ_ESHAPE;
  if (cfg->fmt == SHARQ_HIF4 && D % 128 != 0) return SHARQ_ESHAPE;     // the bf16 emulation tiles D by 128
  if (out_dtype < 0 || out_dtype > 1 || path < 0 || path > 4) return SHARQ_EINVAL;
  for (int i = 0; i < n; ++i)
    if (!ptrs[i] || !aligned16(ptrs[i])) return SHARQ_EINVAL;
  return SHARQ_OK;
}

sharq_status sharq_linear(const sharq_config* cfg, int64_t T, int64_t D, int64_t K, const void* sp_codes,
                          const void* sp_sf, const void* sp_meta, const void* dn_codes, const void* dn_sf,
                          const float* row_scale, const void* w_codes, const void* w_sf_sparse_view,
                          const void* w_sf_dense_view, const float* w_tensor_scale, const void* bias, void* Y,
                          int64_t ldy, int32_t out_dtype, int32_t path, void* workspace, size_t workspace_bytes,
                          void* stream) {
  const void* ptrs[] = {sp_codes, sp_sf, sp_meta, dn_codes, dn_sf, w_codes, w_sf_sparse_view, w_sf_dense_view, Y};
  sharq_status s = check_linear(cfg, D, K, ptrs, T == 0 ? 0 : 9, ldy, out_dtype, path);
  if (s != SHARQ_OK) return s;
  if (T < 0 || T >= (int64_t)1 << 30) return SHARQ_ESHAPE;
  if (T == 0) return SHARQ_OK;
  if (!row_scale || !w_tensor_scale) return SHARQ_EINVAL;
  if (workspace_bytes < linear_workspace_bytes(cfg, T, D, K, 0)) return SHARQ_EWORKSPACE;
  DeviceInfo di{};
  if ((s = device_info(&di)) != SHARQ_OK) return s;
  if (path > 2) return SHARQ_EINVAL;                       // the two-operand combinations go through sharq_linear_paths
  LinearArgs a{T, D, K, sp_codes, sp_sf, sp_meta, dn_codes, dn_sf, nullptr, row_scale, w_codes, w_sf_sparse_view,
               w_sf_dense_view, w_tensor_scale, bias, Y, ldy, out_dtype, path};
  return launch_linear(cfg, a, 0, nullptr, workspace, workspace_bytes, di.sms, di.dev, (cudaStream_t)stream, nullptr);
}

// ---- sharq_prepare_linear --------------------------------------------------------------
sharq_status sharq_prepare_linear(const sharq_config* cfg, const void* x, int64_t T, int64_t K, int64_t ldx,
                                  const void* gamma, const void* beta, const float* x_tensor_scale, void* sp_codes,
                                  void* sp_sf, void* sp_meta, void* dn_codes, void* dn_sf, float* row_scale, int64_t D,
                                  const void* w_codes, const void* w_sf_sparse_view, const void* w_sf_dense_view,
                                  const float* w_tensor_scale, const void* bias, void* Y, int64_t ldy, int32_t out_dtype,
                                  int32_t single_launch, void* workspace, size_t workspace_bytes, void* stream) {
  // single_launch = 0: the two calls it stands for, chained by programmatic dependent launch (measured faster: the
  // prepare kernel runs while the GEMM's CTAs are being scheduled and fill their weight ring); 1: one fused launch
  // when the shape allows it
  sharq_status s = check_cfg(cfg);
  if (s != SHARQ_OK) return s;
  if (single_launch < 0 || single_launch > 1) return SHARQ_EINVAL;
  const bool fusable = single_launch == 1 && cfg->fmt != SHARQ_HIF4 && cfg->mask == SHARQ_MASK_PAIR48 && cfg->layout == SHARQ_LAYOUT_TILED &&
                       cfg->norm != SHARQ_NORM_LAYER && T >= 1 && T <= 8 && K > 0 && K % 256 == 0 && K <= 16384 &&
                       ldx >= K && ldx % 16 == 0 && x && ((uintptr_t)x & 31u) == 0;
  if (!fusable) {
    s = sharq_prepare(cfg, x, T, K, ldx, gamma, beta, x_tensor_scale, sp_codes, sp_sf, sp_meta, dn_codes, dn_sf, row_scale,
                      stream);
    if (s != SHARQ_OK) return s;
    return sharq_linear(cfg, T, D, K, sp_codes, sp_sf, sp_meta, dn_codes, dn_sf, row_scale, w_codes, w_sf_sparse_view,
                        w_sf_dense_view, w_tensor_scale, bias, Y, ldy, out_dtype, 0, workspace, workspace_bytes, stream);
  }
  // the argument checks of the two calls
  if (!sp_codes || !sp_sf || !sp_meta || !dn_codes || !dn_sf || !row_scale) return SHARQ_EINVAL;
  if (cfg->norm != SHARQ_NORM_NONE && !gamma) return SHARQ_EINVAL;
  if (!aligned16(sp_codes) || !aligned16(sp_sf) || !aligned16(sp_meta) || !aligned16(dn_codes) || !aligned16(dn_sf) ||
      (gamma && !aligned16(gamma)))
    return SHARQ_EINVAL;
  const void* ptrs[] = {sp_codes, sp_sf, sp_meta, dn_codes, dn_sf, w_codes, w_sf_sparse_view, w_sf_dense_view, Y};
  if ((s = check_linear(cfg, D, K, ptrs, 9, ldy, out_dtype, 0)) != SHARQ_OK) return s;
  if (!w_tensor_scale) return SHARQ_EINVAL;
  DeviceInfo di{};
  if ((s = device_info(&di)) != SHARQ_OK) return s;
  const PrepParams pp = make_prep_params(cfg, x, T, K, ldx, gamma, beta, x_tensor_scale, sp_codes, sp_sf, sp_meta, dn_codes,
                                         dn_sf, row_scale);
  const FusedArgs fz{&pp, cfg->norm, (int32_t)((K + 1023) / 1024)};
  LinearArgs a{T, D, K, sp_codes, sp_sf, sp_meta, dn_codes, dn_sf, nullptr, row_scale, w_codes, w_sf_sparse_view,
               w_sf_dense_view, w_tensor_scale, bias, Y, ldy, out_dtype, 0};
  return launch_linear(cfg, a, 0, nullptr, workspace, workspace_bytes, di.sms, di.dev, (cudaStream_t)stream, nullptr, &fz);
}

// ---- Table 5 path combinations --------------------------------------------------------------
static bool combo_ok(const sharq_config* cfg, int32_t path) {
  return (path == 3 || path == 4) && cfg->fmt != SHARQ_HIF4 && cfg->mask == SHARQ_MASK_PAIR48;
}

sharq_status sharq_act_sizes_paths(const sharq_config* cfg, int32_t path, int64_t T, int64_t K, size_t* a_codes,
                                   size_t* a_sf, size_t* a_meta, size_t* row_scale) {
  sharq_status s = check_cfg(cfg);
  if (s != SHARQ_OK) return s;
  if (!combo_ok(cfg, path)) return SHARQ_EINVAL;
  if (T < 0 || K <= 0 || K % 256 != 0) return SHARQ_ESHAPE;
  const bool dense = path == 3;
  if (a_codes) *a_codes = (size_t)T * (size_t)(dense ? K / 2 : K / 4);
  if (a_sf) *a_sf = sf_bytes(cfg, T, dense ? sf_cols(cfg->fmt, true, K) : K / 32);
  if (a_meta) *a_meta = dense ? 0 : sf_bytes(cfg, T, K / 16);
  if (row_scale) *row_scale = (size_t)T * sizeof(float);
  return SHARQ_OK;
}

sharq_status sharq_prepare_paths(const sharq_config* cfg, int32_t path, const void* x, int64_t T, int64_t K, int64_t ldx,
                                 const void* gamma, const void* beta, const float* x_tensor_scale, void* a0_codes,
                                 void* a0_sf, void* a0_meta, void* a1_codes, void* a1_sf, void* a1_meta,
                                 float* row_scale, void* stream) {
  sharq_status s = check_cfg(cfg);
  if (s != SHARQ_OK) return s;
  if (!combo_ok(cfg, path)) return SHARQ_EINVAL;
  if (T < 0 || K <= 0 || K % 256 != 0 || ldx < K || ldx % 8 != 0 || K > 100 * 1024) return SHARQ_ESHAPE;
  if (T == 0) return SHARQ_OK;
  if (!x || !a0_codes || !a0_sf || !a1_codes || !a1_sf || !row_scale) return SHARQ_EINVAL;
  if (path == 4 && (!a0_meta || !a1_meta)) return SHARQ_EINVAL;
  if (cfg->norm != SHARQ_NORM_NONE && !gamma) return SHARQ_EINVAL;
  if (!aligned16(x) || !aligned16(a0_codes) || !aligned16(a0_sf) || !aligned16(a1_codes) || !aligned16(a1_sf) ||
      (a0_meta && !aligned16(a0_meta)) || (a1_meta && !aligned16(a1_meta)) || (gamma && !aligned16(gamma)) ||
      (beta && !aligned16(beta)))
    return SHARQ_EINVAL;
  DeviceInfo di{};
  if ((s = device_info(&di)) != SHARQ_OK) return s;
  cudaError_t e = launch_prepare(cfg, x, T, K, ldx, gamma, beta, x_tensor_scale, a0_codes, a0_sf, a0_meta, a1_codes,
                                 a1_sf, row_scale, di.sms, (cudaStream_t)stream, nullptr, 0, nullptr, 0, path, a1_meta);
  return e == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}

sharq_status sharq_linear_paths(const sharq_config* cfg, int32_t path, int64_t T, int64_t D, int64_t K,
                                const void* a0_codes, const void* a0_sf, const void* a0_meta, const void* a1_codes,
                                const void* a1_sf, const void* a1_meta, const float* row_scale, const void* w_codes,
                                const void* w_sf_sparse_view, const void* w_sf_dense_view, const float* w_tensor_scale,
                                const void* bias, void* Y, int64_t ldy, int32_t out_dtype, void* stream) {
  if (!cfg || !combo_ok(cfg, path)) return SHARQ_EINVAL;
  const void* ptrs[] = {a0_codes, a0_sf, a1_codes, a1_sf, w_codes, w_sf_sparse_view, w_sf_dense_view, Y};
  sharq_status s = check_linear(cfg, D, K, ptrs, T == 0 ? 0 : 8, ldy, out_dtype, path);
  if (s != SHARQ_OK) return s;
  if (T < 0 || T >= (int64_t)1 << 30) return SHARQ_ESHAPE;
  if (T == 0) return SHARQ_OK;
  if (!row_scale || !w_tensor_scale) return SHARQ_EINVAL;
  if (path == 4 && (!a0_meta || !a1_meta || !aligned16(a0_meta) || !aligned16(a1_meta))) return SHARQ_EINVAL;
  DeviceInfo di{};
  if ((s = device_info(&di)) != SHARQ_OK) return s;
  LinearArgs a{T, D, K, a0_codes, a0_sf, a0_meta, a1_codes, a1_sf, a1_meta, row_scale, w_codes, w_sf_sparse_view,
               w_sf_dense_view, w_tensor_scale, bias, Y, ldy, out_dtype, path};
  return launch_linear(cfg, a, 0, nullptr, nullptr, 0, di.sms, di.dev, (cudaStream_t)stream, nullptr);
}

sharq_status sharq_linear_grouped(const sharq_config* cfg, int32_t E, const int32_t* offsets, int64_t padded_rows,
                                  int64_t D, int64_t K, const void* sp_codes, const void* sp_sf, const void* sp_meta,
                                  const void* dn_codes, const void* dn_sf, const float* row_scale,
                                  const void* w_codes, const void* w_sf_sparse_view, const void* w_sf_dense_view,
                                  const float* w_tensor_scale, void* Y, int64_t ldy, int32_t out_dtype,
                                  void* workspace, size_t workspace_bytes, void* stream) {
  const void* ptrs[] = {sp_codes, sp_sf, sp_meta, dn_codes, dn_sf, w_codes, w_sf_sparse_view, w_sf_dense_view, Y};
  sharq_status s = check_linear(cfg, D, K, ptrs, 9, ldy, out_dtype, 0);
  if (s != SHARQ_OK) return s;
  if (E <= 0 || !offsets) return SHARQ_EINVAL;
  if (cfg->fmt == SHARQ_HIF4) return SHARQ_EINVAL;
  if (E > 1024 || padded_rows < 0 || padded_rows % 128 != 0 || padded_rows >= (int64_t)1 << 30) return SHARQ_ESHAPE;
  if (!row_scale || !w_tensor_scale) return SHARQ_EINVAL;
  (void)workspace; (void)workspace_bytes;                  // NVFP4 / MXFP4 need none
  if (padded_rows == 0) return SHARQ_OK;
  DeviceInfo di{};
  if ((s = device_info(&di)) != SHARQ_OK) return s;
  LinearArgs a{padded_rows, D, K, sp_codes, sp_sf, sp_meta, dn_codes, dn_sf, nullptr, row_scale, w_codes,
               w_sf_sparse_view, w_sf_dense_view, w_tensor_scale, nullptr, Y, ldy, out_dtype, 0};
  return launch_linear(cfg, a, E, offsets, workspace, workspace_bytes, di.sms, di.dev, (cudaStream_t)stream, nullptr);
}

sharq_status sharq_linear_plan(const sharq_config* cfg, int64_t T, int64_t D, int64_t K, int32_t E, char* buf,
                               size_t n) {
  sharq_status s = check_linear(cfg, D, K, nullptr, 0, D, 0, 0);
  if (s != SHARQ_OK) return s;
  if (!buf || n == 0 || T < 0 || E < 0 || T >= (int64_t)1 << 30) return SHARQ_EINVAL;
  if (E > 0 && (T % 128 != 0 || E > 1024 || cfg->fmt == SHARQ_HIF4)) return SHARQ_ESHAPE;
  DeviceInfo di{};
  if ((s = device_info(&di)) != SHARQ_OK) return s;
  LinearPlan pl{};
  pl.kind = -1;
  LinearArgs a{T, D, K, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
               nullptr, nullptr, nullptr, D, 0, 0};
  if (T > 0) {
    s = launch_linear(cfg, a, E, nullptr, nullptr, 0, di.sms, di.dev, nullptr, &pl);
    if (s != SHARQ_OK) return s;
  }
  static const char* const kinds[] = {"tile", "pair", "grouped-mc", "hif4-bf16", "tile+prepare", "grouped-pair"};
  if (pl.kind < 0) snprintf(buf, n, "none");
  else snprintf(buf, n, "%s bn=%d act_rows=%d splits=%d stages=%d tiles=%lld grid=%lld cluster=%d", kinds[pl.kind],
                pl.bn, pl.act_rows, pl.splits, pl.stages, (long long)pl.tiles, (long long)pl.grid, pl.cluster);
  return SHARQ_OK;
}

sharq_status sharq_act_init(const sharq_config* cfg, int64_t T, int64_t K, void* sp_sf, void* sp_meta, void* dn_sf,
                            void* stream) {
  size_t n_sf = 0, n_meta = 0, n_dn = 0;
  sharq_status s = sharq_act_sizes(cfg, T, K, nullptr, &n_sf, &n_meta, nullptr, &n_dn, nullptr);
  if (s != SHARQ_OK) return s;
  if (cfg->layout != SHARQ_LAYOUT_TILED || T == 0) return SHARQ_OK;
  if (!sp_sf || !sp_meta || !dn_sf) return SHARQ_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  if (cudaMemsetAsync(sp_sf, 0, n_sf, st) != cudaSuccess || cudaMemsetAsync(dn_sf, 0, n_dn, st) != cudaSuccess ||
      cudaMemsetAsync(sp_meta, 0x44, n_meta, st) != cudaSuccess)
    return SHARQ_ECUDA;
  return SHARQ_OK;
}

sharq_status sharq_untile_sf(const void* tiled, int64_t R, int64_t C, void* canonical, void* stream) {
  if (R < 0 || C <= 0 || C % 4 != 0) return SHARQ_ESHAPE;
  if (R == 0) return SHARQ_OK;
  if (!tiled || !canonical) return SHARQ_EINVAL;
  return launch_untile(tiled, R, C, canonical, 0, (cudaStream_t)stream) == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}

sharq_status sharq_untile_meta(const void* tiled, int64_t R, int64_t K, void* canonical, void* stream) {
  if (R < 0 || K <= 0 || K % 256 != 0) return SHARQ_ESHAPE;
  if (R == 0) return SHARQ_OK;
  if (!tiled || !canonical) return SHARQ_EINVAL;
  return launch_untile(tiled, R, K / 16, canonical, 1, (cudaStream_t)stream) == cudaSuccess ? SHARQ_OK : SHARQ_ECUDA;
}

}  // extern "C"
