/* tc_bench.h — MEASUREMENT AIDS of bench.py, kept out of the product contract (include/tc.h).
 *
 * They live in the same library because they must run on the same device, stream and build as the
 * kernels they are compared with; nothing in the hot path uses them.
 */
#ifndef TC_BENCH_H_
#define TC_BENCH_H_

#include "tc.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Measured FP32 peak of the current device: an FFMA-only microbenchmark (16 independent
 * fma.rn.f32 chains per thread, two of the three operands shared by every chain so that the register file is
 * not the limit, 8 CTAs of 256 threads per SM, CUDA events on the context's stream).
 * *tflops = 2 flops x FFMA lane-instructions / time.  This is the denominator the roofline of bench.py
 * quotes beside the nominal SMs x 128 lanes x 2 x clock: the force kernel is bound by the
 * FP32 pipe and its operand supply, not by HBM or tensor throughput (PAPER.md:175 measures "instruction
 * throughput" the same way).  Errors: TC_ESTATE (host-only), TC_EINVAL, TC_ECUDA.                        */
int tc_fp32_peak(tc_ctx* ctx, double* tflops);

/* Option of tc_set_option (include/tc.h) that exists for bench.py only:
 *   "walk_only"   0 (default) or 1: tc_forces walks the tree and builds every interaction list (A1-A3) but
 *                 skips their evaluation; acc and pot are then ZERO, counts and n_tests_total are valid.
 *                 bench.py uses it to report the paper's second metric, the data rate of the tree walk
 *                 (PAPER.md:177).                                                                        */

#ifdef __cplusplus
}
#endif
#endif /* TC_BENCH_H_ */
