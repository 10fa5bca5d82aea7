/*
 * dg_b200_test.h -- TEST-ONLY entry points of libdg_b200.so.  Not part of the product boundary
 * (include/dg_b200.h is); nothing on the hot path calls these.
 */
#ifndef DG_B200_TEST_H
#define DG_B200_TEST_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Self-test of the two device arithmetic helpers the kernels use instead of IEEE division and square
 * root in the flux evaluations of PAPER.md:45-50, 70 (Newton-corrected hardware seeds, no slow-path
 * branches; csrc/dg_internal.h): rcp_out[i] = 1/x[i] and sqrt_out[i] = sqrt(x[i]) for n positive normal
 * doubles.  All three are DEVICE pointers owned by the caller; the call is enqueued on `cuda_stream`
 * (cudaStream_t as void*).  Returns DG_OK, DG_EINVAL (null pointer) or DG_ECUDA (launch failed). */
int dg_selftest_fastmath(const double *x_dev, double *rcp_out_dev, double *sqrt_out_dev, size_t n, void *cuda_stream);

/* FP64 peak microbenchmark for the roofline of bench.py ("measure with an FMA microbenchmark in
 * the same run"): launches `blocks` blocks of 256 threads, each thread running 8 independent chains of
 * double-precision fused multiply-adds, 128 * iters of them per thread, on `cuda_stream`; `out_dev` is a DEVICE
 * array of blocks * 256 doubles that receives the chain sums (so that the work cannot be optimised away);
 * *fma_count (host, may be NULL) = thread-level FMAs executed.  The caller times the launch with CUDA events.
 * Returns DG_OK, DG_EINVAL or DG_ECUDA. */
int dg_fp64_peak(double *out_dev, int blocks, int iters, void *cuda_stream, unsigned long long *fma_count);

#ifdef __cplusplus
}
#endif
#endif /* DG_B200_TEST_H */
