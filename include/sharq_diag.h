/* sharq_diag.h -- diagnostics exported by libsharq.so that are NOT part of the SharQ hot path.
 *
 * sharq_mma_peak_launch: tensor-pipe issue-rate probe.  SURVEY.md 8(d) defines the applicable FP4 tensor peak of
 * the GEMM roofline as "measured on the box by a TMEM-resident MMA issue loop (dense-only, sparse-only)"; this is
 * that loop, and bench.py is its only caller.
 * Launches, on every SM pair, `iters` repetitions of the per-k-block (256 logical k) instruction sequence of the
 * CTA-pair GEMM on shared-memory-resident bytes: mode bit 1 = the 4 dense block-scaled MMAs, bit 2 = the 2 sparse
 * MMAs, bit 4 = the scale-factor / metadata tcgen05.cp copies, bit 8 = pseudo-random operand bits instead of constant
 * bytes (the GPU is power capped: a pipe fed constants runs at higher clocks than one fed data, so the constant-
 * operand rate is an upper bound of the applicable peak and the random-operand rate a lower bound); M = 256, N = 256
 * per pair, no loads, no epilogue.
 * The caller times it (CUDA events): nominal flop per path = 2 * 128 * 256 * 256 * iters * (number of SMs). */
#ifndef SHARQ_DIAG_H_
#define SHARQ_DIAG_H_

#include "sharq.h"

#ifdef __cplusplus
extern "C" {
#endif

sharq_status sharq_mma_peak_launch(int32_t mode, int32_t iters, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* SHARQ_DIAG_H_ */
