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

/* Per-kernel-class timing: between _begin and _end every kernel launch of the library is bracketed by a pair of CUDA
 * events on its stream; _end synchronises the device and returns, per class, the summed event intervals (ms), the
 * ALGORITHMIC flops and bytes of those launches (element-exact: triangular operands and lower-only outputs count what
 * they need, not what the tiles execute; bandwidth classes count the bytes each launch must read or write once) and
 * the number of launches.  Arrays of BTA_KC_COUNT entries; any may be NULL.  Use with BTA_OPT_SERIAL = 1 (one stream)
 * so that the intervals are exclusive.  Process-global (not per ctx); launches inside a CUDA-graph capture are skipped. */
enum {
  BTA_KC_GEMM_BIG = 0,    /* gemm_kernel, 128x128 tiles */
  BTA_KC_GEMM_SMALL = 1,  /* gemm_kernel, 64x64 tiles */
  BTA_KC_GEMM_TINY = 2,   /* gemm_kernel, 32x32 tiles */
  BTA_KC_LEAF = 3,        /* potrf_inv_blocked_kernel: flops 2/3 n^3 */
  BTA_KC_SKINNY = 4,      /* skinny_nt / skinny_nn: bytes = the b x b operand (half if triangular) */
  BTA_KC_CONTRACT = 5,    /* trace_stencil / noise_trace / quad_stencil: bytes = the gathered stencil entries */
  BTA_KC_ASSEMBLE = 6,    /* assemble_*: bytes = the blocks written */
  BTA_KC_OTHER = 7,       /* tips, small products, reductions, scalars */
  BTA_KC_COUNT = 8
};
/* The product of bta_rows_times_block_noalloc (include/bta.h) through the sweeps' own launcher with CALLER-provided
 * scratch `part` (DEVICE, ceil(K/128) * P * J doubles): the existing path the allocation-free variant is tested against. */
BTA_API int bta_rows_times_block(int P, int K, int J, const double* R, int ldr, const double* M, int ldm, int tri,
                                 double alpha, double beta, const double* in, int ldin, double* out, int ldo, double* part,
                                 void* stream);

/* The transposed twin used by the forward sweeps (Algorithm 1 lines 4-5, 9): out[p][j] = beta in[p][j] +
 * alpha sum_k R[p][k] M[j][k] for P <= 16 rows, k restricted to k <= j when tri != 0 (M lower triangular).  DEVICE
 * pointers, row-major; `in` may be NULL when beta == 0 and may alias `out`.  No scratch. */
BTA_API int bta_rows_times_block_t(int P, int J, int K, const double* R, int ldr, const double* M, int ldm, int tri,
                                   double alpha, double beta, const double* in, int ldin, double* out, int ldo,
                                   void* stream);

/* POTRF + TRTRI of one n x n block as the forward sweeps do it (Algorithm 1 line 3, in the
 * inverse-diagonal form of DESIGN.md §5): A (DEVICE, row-major, leading dimension ld, SPD, lower triangle read, strict
 * upper triangle zero as the assembly leaves it) is overwritten by X = chol(A)^-1 (lower triangular); diagL (DEVICE, n
 * doubles, or NULL) receives diag(chol(A)).  T1, T2: DEVICE scratch blocks of the same shape as A, required for n > 128
 * (the blocked recursion over 128 x 128 leaves).  Returns BTA_ERR_NOTSPD on a non-positive pivot (bta_last_pivot = its
 * 1-based row); synchronises the stream.  Kernel-level test hook, not part of the hot path's boundary. */
BTA_API int bta_diag_potrf_inv(bta_ctx* ctx, double* A, int ld, int n, double* T1, double* T2, double* diagL, void* stream);

/* Host-only: the element-exact flop count the timing registers for one GEMM launch (klo/khi/out as in bta_gemm). */
BTA_API double bta_diag_gemm_flop(int M, int N, int K, int klo, int khi, int out);
BTA_API int bta_diag_ktime_begin(void);
BTA_API int bta_diag_ktime_end(double* ms, double* flop, double* bytes, long long* count);

/* Run-time switches of the sweep orchestration (diagnostics and A/B measurements; the defaults are the measured
 * best).  bta_create also reads the environment variables named below once, as initial values.
 *   BTA_OPT_TWIST (BTA_TWIST)          1: two-way elimination, four chains (default); 0: one chain per matrix
 *   BTA_OPT_LANES (BTA_LANES)          1: priority lanes for the small kernels (default); 2: forward only; 0: off
 *   BTA_OPT_SPLIT (BTA_SPLIT)          1: coupled forward step for b <= 1024 (default); 0: off
 *   BTA_OPT_GRAPH (BTA_GRAPH)          -1: CUDA-graph replay for b <= 1024 (default); 0: never; 1: always
 *   BTA_OPT_SERIAL (BTA_SERIAL_CHAINS) 1: both matrices on one stream, single chain -- exclusive per-stage times
 *   BTA_OPT_PIPELINE (BTA_PIPELINE)    1: forward sweeps (b > 1024, factor mode) overlap the first half of the next
 *                                      block's factorisation with the tail of this block's products (default);
 *                                      0: strict block-by-block order
 *   BTA_OPT_TILE_THRESH (BTA_TILE_THRESH), BTA_OPT_TILE_WAVES (BTA_TILE_WAVES): the GEMM tile rule (process-global):
 *                                      launches of fewer 128x128 tiles than the threshold (180) use 64x64 tiles, and
 *                                      (waves = 1) so do launches whose last wave of 128x128 tiles would be mostly empty
 *   BTA_OPT_PDL (BTA_PDL)              programmatic dependent launch of the latency-bound kernels (they start while their
 *                                      predecessor drains and wait at griddepcontrol.wait): 3 (default) the POTRF leaves
 *                                      only, 1 the leaves and the 32x32-tile GEMMs, 2 those GEMMs only, 0 plain launches.
 *                                      Process-global.
 *   BTA_OPT_ROWS (BTA_ROWS)            1 (default): the arrow / right-hand-side rows of the forward steps and the trace
 *                                      contractions of the backward steps run on a third stream per chain (factor
 *                                      mode), off the chain's dependent launch sequence; 0: in line
 *   BTA_OPT_PARTITIONS (BTA_PARTITIONS) >= 2: inla_value_and_grad uses the paper's time-domain partitioning with that
 *                                      many partitions inside the GPU (include/bta.h, "Time-domain partitioning");
 *                                      0 (default): the two-way elimination.  Factor mode only.
 * Returns BTA_ERR_ARG for an unknown option.  Cached CUDA graphs are dropped. */
enum { BTA_OPT_TWIST = 0, BTA_OPT_LANES = 1, BTA_OPT_SPLIT = 2, BTA_OPT_GRAPH = 3, BTA_OPT_SERIAL = 4,
       BTA_OPT_PIPELINE = 5, BTA_OPT_TILE_THRESH = 6, BTA_OPT_TILE_WAVES = 7, BTA_OPT_PARTITIONS = 8, BTA_OPT_PDL = 9,
       BTA_OPT_ROWS = 10 };
BTA_API int bta_set_option(bta_ctx* ctx, int option, int value);
BTA_API int bta_get_option(const bta_ctx* ctx, int option);

#ifdef __cplusplus
}
#endif
#endif /* BTA_DIAG_H_ */
