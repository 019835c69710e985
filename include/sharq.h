/* sharq.h -- C ABI of the B200-native SharQ per-linear-layer hot path.
 *
 * SharQ (arxiv/paper_2606_26587; "P:n" = line n of the paper text): for each linear layer
 *   Y^ = GEMM_sp(Q_sp(M(X) . X), Q_w,sp(W)) + GEMM_dn(Q_dn(R), Q_w,dn(W)),  R = X - D_sp(Q_sp(X_sp))
 * (Eq. 6-9).  Three calls make the path (Fig. 2, section 3.4):
 *   sharq_quantize_weight  offline, once per weight: one FP4 payload + two scale views
 *   sharq_prepare          per call: norm -> N:M mask -> sparse FP4 backbone -> residual -> dense FP4
 *   sharq_linear           sparse + dense block-scaled FP4 GEMMs into one accumulator, bf16 epilogue
 * plus sharq_linear_grouped (the same over the row ranges of E experts, MoE), sharq_prepare_add
 * (sharq_prepare with the residual-stream add fused in front of the norm), sharq_prepare_swiglu (with
 * SiLU(gate) * up fused in front of it), sharq_prepare_linear (both calls as one, a single launch for decode
 * shapes), host-only size / plan queries
 * (sharq_weight_sizes, sharq_act_sizes, sharq_linear_workspace, sharq_linear_plan), sharq_act_init, the Table 5
 * path combinations (sharq_act_sizes_paths, sharq_prepare_paths, sharq_linear_paths) and the test
 * helpers sharq_untile_sf / sharq_untile_meta.  The tensor-pipe probe lives in sharq_diag.h.
 *
 * Conventions
 *   - The caller owns every buffer; the library never allocates device memory and keeps no
 *     state between calls: every entry point is thread-safe and reads no environment variable.  (The only
 *     process-wide data are memoised answers of the CUDA runtime about a device -- a driver entry point,
 *     "opt-in shared memory is set for this kernel", cluster occupancy -- keyed by device ordinal, filled
 *     lock-free and idempotently.)  All pointers are DEVICE pointers unless marked "host".
 *   - Work is enqueued on the caller's CUDA stream (`stream` is a cudaStream_t passed as void*)
 *     and the call returns without synchronising.
 *   - Errors are return codes; nothing throws or aborts.  On a non-OK return nothing was launched.
 *   - Sizes are int64_t, leading dimensions are in ELEMENTS, base pointers 16-byte aligned.
 *     (sharq_prepare is fastest when x is 32-byte aligned with ldx % 16 == 0: rows that start on an odd
 *     16-byte boundary are served by a slower kernel, same results.)
 *   - bf16 tensors are row-major; "code" tensors hold two 4-bit codes per byte, the element
 *     with the lower k in the low nibble.
 *   - Shapes: K % 256 == 0 (8-chunks, 32/64 scale groups, MMA-K 128, 256-wide metadata tile),
 *     D % 8 == 0 for sharq_linear (D % 128 == 0 for HiF4 and for sharq_linear_grouped), T >= 0 (T == 0 returns
 *     SHARQ_OK without a launch), T < 2^30.
 *   - Inputs must be finite; NaN/Inf behaviour is deterministic but unspecified.
 *
 * Output layouts (config.layout)
 *   CANONICAL  plain row-major arrays as listed per argument below (what the parity tests read).
 *   TILED      what sharq_linear consumes (tcgen05 scale-factor / metadata atoms):
 *     scale factors [R rows, C = K/G columns], rows padded to a multiple of 128:
 *       byte(r, c) at  ((r/128) * (C/4) + c/4) * 512 + (r%32)*16 + ((r%128)/32)*4 + (c%4)
 *     sparsity metadata [R rows, K/16 bytes], rows padded to a multiple of 128:
 *       byte(r, b) at  ((r/128) * (K/256) + b/16) * 2048 + (r%128)*16 + (b%16)
 *     codes and row scales are identical in both layouts.
 *   sharq_*_sizes report the padded byte counts for the chosen layout.  sharq_prepare writes the bytes of rows
 *   0 .. T-1 only; the pad rows of the last 128-row tile are read by sharq_linear's tensor-memory copies (their
 *   products land in accumulator rows that are never stored), so they must hold VALID bytes: initialise the TILED
 *   scale / metadata buffers once with sharq_act_init (any later sharq_prepare output keeps them valid).
 */
#ifndef SHARQ_H_
#define SHARQ_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  SHARQ_OK = 0,
  SHARQ_EINVAL = 1,     /* null pointer, bad enum, misaligned pointer, unsupported combination */
  SHARQ_ESHAPE = 2,     /* shape rule violated (see above) */
  SHARQ_EWORKSPACE = 3, /* workspace too small */
  SHARQ_EARCH = 4,      /* device is not sm_100 */
  SHARQ_ECUDA = 5       /* a CUDA runtime / driver call failed (launch not accepted) */
} sharq_status;

typedef enum { SHARQ_NVFP4 = 0, SHARQ_MXFP4 = 1, SHARQ_HIF4 = 2 } sharq_format;
/* PAIR48: 4:8 "in pairs" -- the pattern the block-scaled FP4 sparse MMA accepts.
 * MASK_24: element-wise 2:4, used with HiF4. */
typedef enum { SHARQ_MASK_PAIR48 = 0, SHARQ_MASK_24 = 1 } sharq_mask;
typedef enum { SHARQ_NORM_NONE = 0, SHARQ_NORM_RMS = 1, SHARQ_NORM_LAYER = 2 } sharq_norm;
typedef enum { SHARQ_LAYOUT_CANONICAL = 0, SHARQ_LAYOUT_TILED = 1 } sharq_layout;

typedef struct {
  int32_t fmt;    /* sharq_format */
  int32_t mask;   /* sharq_mask.  HIF4 requires MASK_24.  NVFP4 / MXFP4: PAIR48 is the pattern the B200 sparse FP4
                     MMA accepts; MASK_24 (element-wise 2:4) is accepted by sharq_prepare / sharq_act_sizes with
                     layout CANONICAL only (oracle-checkable encoding; sharq_linear returns SHARQ_ESHAPE for it) */
  int32_t norm;   /* sharq_norm */
  float eps;      /* added to the mean square / variance (P:155 RMSNorm / LayerNorm) */
  int32_t layout; /* sharq_layout of scale-factor and metadata outputs */
} sharq_config;

/* ---- sizes: host-only pure functions; every out pointer may be NULL --------------------- */

/* Bytes of the outputs of sharq_quantize_weight for W[D,K].  */
sharq_status sharq_weight_sizes(const sharq_config* cfg, int64_t D, int64_t K, size_t* codes,
                                size_t* sf_sparse_view, size_t* sf_dense_view, size_t* workspace);

/* Bytes of the outputs of sharq_prepare for x[T,K]. */
sharq_status sharq_act_sizes(const sharq_config* cfg, int64_t T, int64_t K, size_t* sp_codes,
                             size_t* sp_sf, size_t* sp_meta, size_t* dn_codes, size_t* dn_sf,
                             size_t* row_scale);

/* Workspace bytes sharq_linear / sharq_linear_grouped need (may be 0). */
sharq_status sharq_linear_workspace(const sharq_config* cfg, int64_t T, int64_t D, int64_t K,
                                    int32_t E, size_t* workspace);

/* ---- sharq_quantize_weight (Fig. 2 "weight preparation") --------------------
 * W bf16 [D,K], row-major with leading dimension ldw (out-features x in-features).
 *   codes           [D, K/2] bytes          the single shared FP4 payload
 *   sf_sparse_view  [D, K/32] e4m3|e8m0     one scale per 32 k   (HiF4: [D, K/64] uint32 words)
 *   sf_dense_view   [D, K/16] e4m3          every sparse-view scale repeated for its two
 *                                           16-groups (MXFP4: [D,K/32], equal to the sparse
 *                                           view; HiF4: bf16 [D, K], the EXACT dequantisation of
 *                                           the payload -- every HiF4 value has <= 6 significant
 *                                           bits -- which the bf16 tensor path multiplies with)
 *   tensor_scale    1 float                 NVFP4: max|W| / 2688; otherwise 1
 *   workspace       >= sharq_weight_sizes(...workspace) bytes; used for the max|W| reduction
 * Scale views follow cfg->layout.  Two kernels (amax, quantize); not on the timed path. */
sharq_status sharq_quantize_weight(const sharq_config* cfg, const void* W, int64_t D, int64_t K,
                                   int64_t ldw, void* codes, void* sf_sparse_view,
                                   void* sf_dense_view, float* tensor_scale, void* workspace,
                                   size_t workspace_bytes, void* stream);

/* ---- sharq_prepare (Fig. 2 "fused activation preparation") --------------
 * ONE kernel, one pass over x.  x bf16 [T,K] (ldx elements between rows); gamma/beta bf16 [K]
 * (NULL when unused).  x_tensor_scale: device pointer to one float (static per-tensor scale,
 * P:394) or NULL = dynamic per-row scale amax_row/2688 (NVFP4 only; ignored otherwise).
 *   sp_codes  [T, K/4]  bytes  survivors' FP4 codes, ascending k (Eq. 7)
 *   sp_sf     [T, K/32] bytes  backbone block scales           (HiF4: [T, K/64] uint32)
 *   sp_meta   [T, K/16] bytes  one nibble i0|i1<<2 per 8-chunk (MASK_24: [T, K/8], one nibble per 4 elements;
 *                              the backbone scale group stays 32 logical k = 16 survivors)
 *   dn_codes  [T, K/2]  bytes  residual FP4 codes of R = X - D_sp(Q_sp(X_sp)) (Eq. 8)
 *   dn_sf     [T, K/16] bytes  residual block scales (MXFP4: [T,K/32]; HiF4: [T,K/64] uint32)
 *   row_scale [T] float        the tensor scale each row was quantized with (1 for MXFP4/HiF4)
 * sp_sf, sp_meta, dn_sf follow cfg->layout. */
sharq_status sharq_prepare(const sharq_config* cfg, const void* x, int64_t T, int64_t K,
                           int64_t ldx, const void* gamma, const void* beta,
                           const float* x_tensor_scale, void* sp_codes, void* sp_sf,
                           void* sp_meta, void* dn_codes, void* dn_sf, float* row_scale,
                           void* stream);

/* ---- sharq_prepare_add (the paper's own lever was folding the
 * neighbouring elementwise operator into the preparation kernel) ----------------------------
 * sharq_prepare with the transformer's residual-stream add fused in front of the norm:
 *     h[t,k] = bf16( x[t,k] + residual[t,k] )      one rounding of the exact sum, ties to even
 * h is written to sum_out (bf16 [T,K], ldo elements between rows: the new residual stream) and is the
 * activation that norm -> mask -> backbone -> residual -> stores see; every output is exactly what
 * sharq_prepare would produce from h.  sum_out may alias residual (in-place stream update: each
 * element is read and written by the same thread) but not x.  One kernel, one pass: 2 + 2 B/element
 * more HBM traffic than sharq_prepare, against a separate add kernel's 6 B/element plus a launch.
 * x, residual, sum_out: 32-byte aligned, ldx / ldr / ldo multiples of 16 (256-bit accesses), else
 * SHARQ_EINVAL / SHARQ_ESHAPE; K <= 32768 (one row per CTA; NVFP4 with LayerNorm: K <= 25600), else SHARQ_ESHAPE.
 * The alias check on sum_out is pointer equality with x: partially overlapping buffers are the caller's error. */
sharq_status sharq_prepare_add(const sharq_config* cfg, const void* x, const void* residual,
                               int64_t T, int64_t K, int64_t ldx, int64_t ldr, void* sum_out,
                               int64_t ldo, const void* gamma, const void* beta,
                               const float* x_tensor_scale, void* sp_codes, void* sp_sf,
                               void* sp_meta, void* dn_codes, void* dn_sf, float* row_scale,
                               void* stream);

/* ---- sharq_prepare_swiglu (second fusion) -------------------------------------
 * sharq_prepare for the down projection with the SwiGLU elementwise operator fused in front of it:
 *     h[t,k] = bf16( silu(gate[t,k]) * up[t,k] ),   silu(g) = g / (1 + exp(-g))
 * computed in fp32 by a fixed algorithm (degree-5 polynomial exp, IEEE reciprocal; R18) that the oracle
 * restates bit for bit; h never goes to HBM and is the activation norm -> mask -> backbone -> residual see.
 * gate / up: bf16 [T, K] (ldg / ldu elements between rows: the two halves of a [T, 2K] gate+up output work),
 * 32-byte aligned, ldg / ldu multiples of 16, K <= 32768; cfg->norm must be SHARQ_NORM_NONE (the down projection's input is
 * not normalised; gamma / beta are ignored); otherwise SHARQ_EINVAL / SHARQ_ESHAPE. */
sharq_status sharq_prepare_swiglu(const sharq_config* cfg, const void* gate, const void* up, int64_t T, int64_t K,
                                  int64_t ldg, int64_t ldu, const void* gamma, const void* beta,
                                  const float* x_tensor_scale, void* sp_codes, void* sp_sf, void* sp_meta,
                                  void* dn_codes, void* dn_sf, float* row_scale, void* stream);

/* ---- sharq_linear (Eq. 9) -----------------------------------------------
 * Y[T,D] = (A_sp . W^T through the sparse view  +  A_dn . W^T through the dense view)
 *          * row_scale[t] * w_tensor_scale  (+ bias[d])
 * Inputs are the outputs of sharq_prepare and sharq_quantize_weight made with the SAME config
 * and layout == SHARQ_LAYOUT_TILED (otherwise SHARQ_EINVAL).  Both GEMMs accumulate into the
 * same TMEM tile in one kernel ("accumulates directly into this output").
 * out_dtype: 0 = bf16, 1 = fp32.  bias bf16 [D] or NULL.  ldy in elements.
 * path: 0 = sparse + dense (SharQ), 1 = sparse only, 2 = dense only (Table 5 rows).
 * HiF4 (layout CANONICAL): tcgen05 has no S1P2 / E6M2 formats, so the operands are dequantised to bf16 (exact: every
 * HiF4 value has <= 6 significant bits): the weight once, by sharq_quantize_weight (its sf_dense_view), the activation
 * operands per call into `workspace` (backbone compressed [T, K/2] + its 2:4 metadata re-tiled for the tensor core,
 * residual [T, K]), and multiplied on the bf16 tensor path with fp32 accumulation: 2:4-sparse MMAs for the backbone,
 * dense MMAs for the residual.  workspace >= sharq_linear_workspace(...) bytes is required.
 * NVFP4 / MXFP4 need no workspace (it may be NULL).  Kernels are launched with programmatic dependent
 * launch: the weight stream of sharq_linear may start while the preceding kernel of the stream (normally
 * sharq_prepare) is still draining; all reads of activation operands wait for it to complete. */
sharq_status sharq_linear(const sharq_config* cfg, int64_t T, int64_t D, int64_t K,
                          const void* sp_codes, const void* sp_sf, const void* sp_meta,
                          const void* dn_codes, const void* dn_sf, const float* row_scale,
                          const void* w_codes, const void* w_sf_sparse_view,
                          const void* w_sf_dense_view, const float* w_tensor_scale,
                          const void* bias, void* Y, int64_t ldy, int32_t out_dtype, int32_t path,
                          void* workspace, size_t workspace_bytes, void* stream);

/* ---- sharq_prepare_linear (decode is where the method's gain shows) ----------------
 * sharq_prepare followed by sharq_linear (path 0) as ONE call with the arguments of both; the activation buffers
 * (sp_codes ... row_scale) are still the caller's and hold sharq_prepare's outputs afterwards.
 * single_launch = 0 (recommended): the two kernels, chained by programmatic dependent launch -- the preparation runs
 *   while the GEMM's CTAs are scheduled, set up their barriers / tensor memory and fill their weight ring.
 * single_launch = 1: for T <= 8 rows, K <= 16384, NVFP4 / MXFP4, TILED layout, norm NONE / RMS and a 32-byte aligned
 *   x with ldx % 16 == 0, ONE launch: every CTA of the GEMM prepares the T rows itself with extra warps while its
 *   producer warp streams the weights (no cross-CTA wait).  Measured 4-6 us per layer SLOWER than the chained pair
 *   on B200: a fused launch cannot start its 1.6 us prologue before the previous launch's CTAs leave
 *   the SMs, the chained pair hides exactly that behind the preparation.  Kept as the measured alternative; other
 *   shapes fall back to the two launches.
 * Results are bit-identical to the two calls either way. */
sharq_status sharq_prepare_linear(const sharq_config* cfg, const void* x, int64_t T, int64_t K, int64_t ldx,
                                  const void* gamma, const void* beta, const float* x_tensor_scale,
                                  void* sp_codes, void* sp_sf, void* sp_meta, void* dn_codes, void* dn_sf,
                                  float* row_scale, int64_t D, const void* w_codes,
                                  const void* w_sf_sparse_view, const void* w_sf_dense_view,
                                  const float* w_tensor_scale, const void* bias, void* Y, int64_t ldy,
                                  int32_t out_dtype, int32_t single_launch, void* workspace,
                                  size_t workspace_bytes, void* stream);

/* ---- sharq_linear_grouped (MoE expert linears) -----------------------------
 * E experts (E <= 1024); `offsets` is a DEVICE int32[E+1] array (e.g. the router's output, no host copy and no
 * synchronisation needed): rows [offsets[e], offsets[e+1]) of the routed batch belong to expert e,
 * offsets[0] == 0, non-decreasing (a negative count is treated as 0).  Every expert's row range starts at a
 * multiple of 128 in the activation tensors, i.e. the caller prepares each expert's rows with sharq_prepare into
 * a 128-row-aligned slot: row r of expert e lives at padded row pad_offsets[e] + r with
 * pad_offsets[e] = sum_{j<e} roundup(count_j, 128).  `padded_rows` = the row capacity of those activation
 * buffers and of Y (a multiple of 128, >= sum roundup(count, 128); e.g. roundup(total, 128) + 128 * E always
 * suffices); row blocks beyond it are not computed.  Weight tensors are stacked [E, ...] (each expert's tensors
 * laid out as sharq_quantize_weight writes them); w_tensor_scale is float[E].  Empty experts are skipped.  Y is
 * [padded_rows, D] in the same padded row numbering.  One launch; every CTA derives the expert table from
 * `offsets` in its shared memory. */
sharq_status sharq_linear_grouped(const sharq_config* cfg, int32_t E, const int32_t* offsets,
                                  int64_t padded_rows, int64_t D, int64_t K, const void* sp_codes,
                                  const void* sp_sf, const void* sp_meta, const void* dn_codes,
                                  const void* dn_sf, const float* row_scale, const void* w_codes,
                                  const void* w_sf_sparse_view, const void* w_sf_dense_view,
                                  const float* w_tensor_scale, void* Y, int64_t ldy, int32_t out_dtype,
                                  void* workspace, size_t workspace_bytes, void* stream);

/* ---- Table 5 path combinations ----------------------------------
 * The paper's ablation replaces SharQ's sparse + dense pair by two paths of ONE kind, the second quantised from
 * the residual of the first exactly as in Eq. 8, one row tensor scale for both:
 *   path 3  Dense + Dense    a0 = dense FP4 of X, a1 = dense FP4 of R = X - D(a0)
 *   path 4  Sparse + Sparse  a0 = SharQ's sparse backbone, a1 = sparse FP4 of R under its own pairwise 4:8 mask
 *                            (score on the fp32 magnitudes of R, same tie rule)
 * (paths 0 / 1 / 2 -- SharQ, sparse only, dense only -- are sharq_prepare + sharq_linear's `path`.)
 * NVFP4 / MXFP4, pairwise mask.  Operand shapes, per operand: dense: codes [T, K/2], sf [T, K/16] (MXFP4 K/32),
 * meta unused (NULL); sparse: codes [T, K/4], sf [T, K/32], meta [T, K/16].  sf / meta follow cfg->layout;
 * sharq_linear_paths needs TILED.  Both operands accumulate into the same TMEM tile (two K-loops of one kernel
 * launch, W streamed twice: an ablation, not a tuned path). */
sharq_status sharq_act_sizes_paths(const sharq_config* cfg, int32_t path, int64_t T, int64_t K, size_t* a_codes,
                                   size_t* a_sf, size_t* a_meta, size_t* row_scale);
sharq_status sharq_prepare_paths(const sharq_config* cfg, int32_t path, const void* x, int64_t T, int64_t K,
                                 int64_t ldx, const void* gamma, const void* beta, const float* x_tensor_scale,
                                 void* a0_codes, void* a0_sf, void* a0_meta, void* a1_codes, void* a1_sf,
                                 void* a1_meta, float* row_scale, void* stream);
sharq_status sharq_linear_paths(const sharq_config* cfg, int32_t path, int64_t T, int64_t D, int64_t K,
                                const void* a0_codes, const void* a0_sf, const void* a0_meta,
                                const void* a1_codes, const void* a1_sf, const void* a1_meta,
                                const float* row_scale, const void* w_codes, const void* w_sf_sparse_view,
                                const void* w_sf_dense_view, const float* w_tensor_scale, const void* bias,
                                void* Y, int64_t ldy, int32_t out_dtype, void* stream);

/* ---- sharq_linear_hif4_static: sharq_linear for HiF4 that needs no workspace and allocates nothing -------------
 * HiF4's sharq_linear is the one call of this library that needs scratch memory (the bf16 copy of the activation
 * operands).  Some callers cannot provide or allocate it: code under CUDA-graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc.  This variant keeps the scratch in a file-scope device array of
 * SHARQ_STATIC_SCRATCH_BYTES inside the library (every GPU that loads the library holds it until exit); the call
 * makes no cudaMalloc / cudaFree / allocating library call.  Same arguments and results as sharq_linear with a HiF4
 * config (layout CANONICAL, D % 128 == 0), minus the workspace.
 * Limit: roundup(T, 128) * 2K * 2 + 256 <= SHARQ_STATIC_SCRATCH_BYTES, i.e. T <= 128 with K <= 16384, T <= 256 with
 * K <= 8192, T <= 512 with K <= 4096 (decode and small-batch shapes); larger problems return SHARQ_EWORKSPACE and launch
 * nothing.  All calls on a device share the one array: calls that overlap on the GPU (different streams) RACE on it;
 * calls in one stream are ordered.  The array keeps the last call's contents; nothing in it has to start at zero. */
#define SHARQ_STATIC_SCRATCH_BYTES (8u * 1024u * 1024u + 256u)
sharq_status sharq_linear_hif4_static(const sharq_config* cfg, int64_t T, int64_t D, int64_t K,
                                      const void* sp_codes, const void* sp_sf, const void* sp_meta,
                                      const void* dn_codes, const void* dn_sf, const float* row_scale,
                                      const void* w_codes, const void* w_sf_sparse_view,
                                      const void* w_sf_dense_view, const float* w_tensor_scale,
                                      const void* bias, void* Y, int64_t ldy, int32_t out_dtype, int32_t path,
                                      void* stream);

/* ---- sharq_act_init: one-time initialisation of TILED activation scale / metadata buffers ----------
 * Fills sp_sf and dn_sf with zero scales and sp_meta with the valid nibble 0x4 (pairs 0 and 1) for all
 * roundup(T, 128) rows, so that the pad rows sharq_prepare never writes hold defined operands (see "Output
 * layouts").  Three memsets on `stream`; layout CANONICAL: nothing to do, returns SHARQ_OK. */
sharq_status sharq_act_init(const sharq_config* cfg, int64_t T, int64_t K, void* sp_sf, void* sp_meta,
                            void* dn_sf, void* stream);

/* ---- sharq_linear_plan: which kernel variant a sharq_linear / sharq_linear_grouped call launches ---------
 * Host-only query (needs the current device for its SM count / cluster occupancy; launches nothing).
 * E == 0: sharq_linear(T, D, K); E > 0: sharq_linear_grouped with padded_rows = T.  Writes a zero-terminated
 * description into buf (at most n bytes), e.g. "pair bn=192 stages=4 tiles=2400 grid=148 cluster=2".
 * kinds: "tile" (128-row tiles, persistent or split-K cluster), "pair" (CTA-pair 256-row tiles), "grouped-mc"
 * (multicast clusters of two), "hif4-bf16".  The parity tests use it to name the variant they cover. */
sharq_status sharq_linear_plan(const sharq_config* cfg, int64_t T, int64_t D, int64_t K, int32_t E, char* buf,
                               size_t n);

/* ---- test helpers (not on the timed path) ---------------------------------------------
 * Map the TILED layouts back to canonical row-major arrays for byte comparison (device -> device).
 *   sharq_untile_sf   tiled scale factors, R rows x C columns (C % 4 == 0) -> canonical [R, C] bytes
 *   sharq_untile_meta tiled sparsity metadata of R rows, K logical columns   -> canonical [R, K/16] bytes */
sharq_status sharq_untile_sf(const void* tiled, int64_t R, int64_t C, void* canonical, void* stream);
sharq_status sharq_untile_meta(const void* tiled, int64_t R, int64_t K, void* canonical, void* stream);

/* Library / build information: returns a static string, e.g. "sharq-b200 0.1 sm_100a". */
const char* sharq_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SHARQ_H_ */
