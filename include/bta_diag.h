/* bta_diag.h -- measurement and diagnostic entry points of libbta_b200.so.  NOT part of the hot path's boundary
 * (that is include/bta.h): bench.py uses bta_fp64_peak / bta_gemm for the roofline denominators and the isolated
 * b x b x b product; `python -m paper_2605_06392_b200.diagnostics` uses the per-CTA timeline. */
#ifndef BTA_DIAG_H_
#define BTA_DIAG_H_

#include "bta.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Register-resident issue loops on all SMs, returning achieved FP64
 * TFLOP/s of `mma.sync.m8n8k4.f64` (kind 0) or DFMA (kind 1) -- the FP64 roofline denominators. */
BTA_API int bta_fp64_peak(int kind, int iters, double* tflops, double* ms, void* stream);
/* Plain C = alpha op(A) op(B) + beta C through the library's DMMA GEMM (DEVICE pointers, row-major);
 * mode: 0 NN, 1 NT, 2 TN; klo/khi/out as in csrc/common.cuh (0 = full). */
BTA_API int bta_gemm(int mode, int M, int N, int K, double alpha, const double* A, int lda, const double* B, int ldb,
             double beta, double* C, int ldc, int klo, int khi, int out, void* stream);

/* Diagnostic (not on the hot path): one record {start ns, end ns, smid | tile << 16 | mode << 28, k-range | M << 32}
 * per GEMM CTA into buf[cap][4] (DEVICE memory, caller-owned, must outlive the tracing); buf = NULL switches it off.
 * Both calls synchronise the device.  bta_debug_cta_trace_count returns the number of CTAs seen since it was armed. */
BTA_API int bta_debug_cta_trace(unsigned long long* buf, unsigned int cap);
BTA_API int bta_debug_cta_trace_count(unsigned int* n);

/* Run-time switches of the sweep orchestration (diagnostics and A/B measurements; the defaults are the measured
 * best).  bta_create also reads the environment variables named below once, as initial values.
 *   BTA_OPT_TWIST (BTA_TWIST)          1: two-way elimination, four chains (default); 0: one chain per matrix
 *   BTA_OPT_LANES (BTA_LANES)          1: priority lanes for the small kernels (default); 2: forward only; 0: off
 *   BTA_OPT_SPLIT (BTA_SPLIT)          1: coupled forward step for b <= 1024 (default); 0: off
 *   BTA_OPT_GRAPH (BTA_GRAPH)          -1: CUDA-graph replay for b <= 1024 (default); 0: never; 1: always
 *   BTA_OPT_SERIAL (BTA_SERIAL_CHAINS) 1: both matrices on one stream, single chain -- exclusive per-stage times
 *   BTA_OPT_PIPELINE (BTA_PIPELINE)    1: forward sweeps overlap the next block's factorisation with the tail of
 *                                      this block's products (default); 0: strict block-by-block order
 * Returns BTA_ERR_ARG for an unknown option.  Cached CUDA graphs are dropped. */
enum { BTA_OPT_TWIST = 0, BTA_OPT_LANES = 1, BTA_OPT_SPLIT = 2, BTA_OPT_GRAPH = 3, BTA_OPT_SERIAL = 4,
       BTA_OPT_PIPELINE = 5 };
BTA_API int bta_set_option(bta_ctx* ctx, int option, int value);
BTA_API int bta_get_option(const bta_ctx* ctx, int option);

#ifdef __cplusplus
}
#endif
#endif /* BTA_DIAG_H_ */
