/* ctaux_testing.h -- test and measurement helpers exported by libctaux_b200.so BESIDE the walker boundary
 * (include/ctaux.h).  Nothing here is part of the hot path's interface: tests use these entry points to reach the
 * library's FP64 tensor-core GEMM tile and its device Philox directly, bench.py to measure the FP64 issue-rate peak.
 * Same conventions as ctaux.h: plain pointers (HOST or DEVICE as stated), 0 or a negative CTAUX_E* code. */
#ifndef CTAUX_TESTING_H_
#define CTAUX_TESTING_H_

#include "ctaux.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Stand-alone FP64 GEMM through the library's TMA-staged DMMA tile kernel (the kernel S2 / S4 / S5 use, PAPER.md:226,
 * 373): C (MxN, ldc) = beta*C + alpha * A (MxK, lda) * B, all column-major DEVICE pointers, K >= 1.
 * A: lda a multiple of 8 and >= M rounded up to 8 ("M-major" operand).  b_nmajor = 0: B is K x N with leading dimension
 * ldb (a multiple of 4, >= K rounded up to 4; the "K-major" right operand, e.g. N in the candidate-row product);
 * b_nmajor = 1: B points to B^T stored column-major, N x K with ldb a multiple of 8 and >= N rounded up to 8 (the
 * "N-major" right operand, e.g. V in the flush).  Builds two tensor maps per call and synchronises the stream. */
int ctaux_dgemm(void* stream, int32_t M, int32_t N, int32_t K, double alpha, const double* A, int32_t lda,
                const double* B, int32_t ldb, double beta, double* C, int32_t ldc, int32_t b_nmajor);

/* Issue-rate peak of the FP64 pipes on the current device, TFLOP/s.  which = 0: DMMA.8x8x4 (mma.sync m8n8k4 f64, the
 * tensor path the GEMM tiles use), 1: DFMA.  Two CTAs of 256 threads per SM, 16 independent accumulators per warp /
 * thread, CUDA events.  The roofline ceiling bench.py prints beside the cuBLAS DGEMM figure. */
int ctaux_probe_fp64(int32_t which, double* tflops);

/* Philox4x32-10 evaluated ON THE DEVICE for n (counter, key) pairs (pin P12: device generator = oracle generator).
 * ctr: HOST [n][4], key: HOST [n][2], out: HOST [n][4]. */
int ctaux_debug_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out, int32_t n);

#ifdef __cplusplus
}
#endif
#endif /* CTAUX_TESTING_H_ */
