/*
 * nspt_debug.h -- diagnostics of libnspt that are NOT part of the method's boundary (include/nspt.h): kernel selection
 * for cross-checks and experiments, per-stage device timing, the FP64 tensor-pipe probe that supplies the roofline
 * denominator, and the launch counter the benchmark reports.  Same conventions as nspt.h (int return codes, current
 * device's context).
 */
#ifndef NSPT_DEBUG_H
#define NSPT_DEBUG_H

#include "nspt.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Select the kernel of the mode-wise matrix product (Step 3):
 *  -1 = automatic (default): the INT8 tensor-core path where it is measured faster and its error stays far below the
 *       tolerance (16 <= L <= 128 and N >= 192; from N >= 160 for the staple, the exponential and the link update where
 *       L >= 32), the FP64 tensor-pipe kernel elsewhere,
 *   0 = reference kernel (one thread per output element, plain double FMAs; cross-check only),
 *   1 = FP64 tensor-pipe kernel (DMMA, TMA-fed, 3-multiplication complex product) everywhere,
 *   2 = INT8 tensor-core path wherever it exists (L >= 16): the forward transform records the largest element of every
 *       mode, one pass cuts both spectra into seven int8 slices per plane (fixed point relative to that maximum), a
 *       persistent tcgen05.mma.kind::i8 kernel forms the exact INT32 sums in TMEM and recombines them in FP64
 *       (SURVEY.md 8f NEXT-3), with the scaling / accumulating / conjugate-transposed epilogues the staple and the exponential
 *       need.  Needs extra workspace (nspt_workspace_bytes reports it for the variant that is selected when it is called),
 *   3 = persistent warp-specialised FP64 tensor-pipe kernel (measured slower than 1; kept as a cross-check),
 *   4 = as 2 with every tile on a CTA pair (tcgen05.mma.cta_group::2, M = 256). */
int nspt_set_gemm_variant(int variant);

/* Select the convolution algorithm of nspt_series_mul[_batched]: 0 = automatic (default), 1 = FFT-CONV,
 * 2 = Naive-CONV (eq. 2.5 evaluated directly, one launch of the tensor-pipe kernel with the K dimension
 * concatenated over the order index; no transforms, no workspace), 3 = FFT-CONV fused into one launch (one CTA per output
 * series, transforms and product in shared memory; only where both operand blocks fit: 2 N (L + 1) + 256 complex128 <= 200 KB;
 * elsewhere the general FFT-CONV runs).  The automatic choice takes 2 for very low orders of small matrices and 3 while
 * N^3 L <= 150000 (N = 12 at N_trunc = 31, N = 16 at N_trunc = 15).  Both read their inputs while they write their output, so a call whose output aliases an input uses the general
 * FFT-CONV whatever is selected here. */
int nspt_set_conv_algorithm(int algorithm);

/* Per-stage device timing.  After nspt_profile(1) every kernel the library launches is
 * bracketed by CUDA events on the library stream; nspt_profile_read synchronises the stream,
 * and for stage = 0 forward transforms, 1 mode-wise matrix products, 2 inverse transforms,
 * 3 re-truncation transforms, 4 other (dagger, force, scaling), 5 block polynomials of the series
 * exponential, 6 int8 slicing passes of the INT8 path returns the summed milliseconds and the number of
 * launches since the last read, then resets the counters. */
int nspt_profile(int enable);
int nspt_profile_read(int stage, double* ms, long long* launches);

/* Measure the FP64 tensor-pipe peak of the current device (TFLOP/s) with a DMMA.8x8x4 chain
 * microbenchmark on the legacy default stream (about 50 ms, synchronous).  This is the roofline
 * denominator for the mode-wise matrix product; it is not part of the hot path. */
int nspt_probe_fp64_peak(double* tflops);

/* Total kernels launched by the library since it was loaded. */
long long nspt_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* NSPT_DEBUG_H */
