/* bta.h -- C-ABI boundary of the B200-native BTA / INLA library (libbta_b200.so).
 *
 * One thing is built behind this boundary: the exact value f(theta) and exact reverse-mode gradient of
 * the INLA objective over a block-tridiagonal-arrowhead (BTA) precision matrix -- the data-parallel hot
 * path of ADELIA (arxiv/paper_2605_06392).  Citations are PAPER.md:<line> (+ equation / algorithm) and
 * DESIGN.md readings R<n>.  Every call runs hand-written sm_100a kernels; there is no CPU fallback:
 * bta_create fails with BTA_ERR_NODEVICE when no compute-capability-10.x device is present.
 *
 * Conventions
 *   - All matrices are FP64, row-major.  "host" / "device" is stated per pointer.
 *   - Notation: nt diagonal blocks D_i (b x b), sub-diagonal blocks B_i = Q[i+1, i]
 *     (b x b, i < nt-1), arrow blocks C_i = Q[T, i] (a x b), tip T (a x a); N = nt*b + a.  b = k*ns,
 *     ns = g*g grid nodes, k response variables.  Latent ordering (R6): index = t*b + v*ns + s, the a
 *     fixed effects last.
 *   - Device block arrays:  D[t][i][j] = Q[t*b+i, t*b+j];  B[t][i][j] = Q[(t+1)*b+i, t*b+j];
 *     C[t][p][j] = Q[nt*b+p, t*b+j];  T[p][q];  rhs[t*b+i], tip entries last (N doubles).
 *   - Ownership: the caller owns every large device buffer (blocks, workspace, rhs) -- typically
 *     torch tensors' data_ptr(); the library allocates only the theta-independent model data
 *     (bta_create) and small scratch.  `stream` is a cudaStream_t passed as void*.
 *   - Return value: 0 on success; BTA_ERR_* (> 0) otherwise; BTA_ERR_NOTSPD means a non-positive pivot
 *     was met on the device (the 1-based global row is reported by bta_last_error / bta_last_pivot).
 *     Calls that return scalars to host memory synchronise `stream` before returning.
 */
#ifndef BTA_H_
#define BTA_H_

#include <stddef.h>
#include <stdint.h>

/* The library is built with -fvisibility=hidden: only the entry points declared here (and in bta_diag.h) are exported. */
#if defined(__GNUC__)
#define BTA_API __attribute__((visibility("default")))
#else
#define BTA_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

enum {
  BTA_OK = 0,
  BTA_ERR_ARG = 1,           /* invalid argument (text in bta_last_error) */
  BTA_ERR_CUDA = 2,          /* a CUDA runtime call or kernel failed */
  BTA_ERR_NODEVICE = 3,      /* no sm_100-class device: the library has no fallback */
  BTA_ERR_NOTSPD = 4,        /* non-positive pivot in a Cholesky step */
  BTA_ERR_UNIMPLEMENTED = 5
};

enum { BTA_PRIOR = 0, BTA_COND = 1 }; /* which matrix: Q_p (BT, no arrow coupling) or Q_c (full BTA) */

typedef struct bta_ctx bta_ctx; /* opaque: model shape, theta-independent observation aggregates, scratch */

/* Model shape (BASELINE.json configs).  d = 3k + k(k-1)/2 + k hyperparameters,
 * ordered (R13): theta_{1,1..3}, ..., theta_{k,1..3}, lambda_21, lambda_31, lambda_32, ..., log tau_1..k. */
typedef struct {
  int32_t nt;        /* time blocks (paper's n) */
  int32_t g;         /* grid side, ns = g*g */
  int32_t k;         /* response variables */
  int32_t a;         /* arrow width = fixed effects (multiple of k; a/k covariates per observation row, R14) */
  double h;          /* grid spacing: C = h^2 I (R3) */
  double fixed_prec; /* prior precision of the fixed effects (R5) */
} bta_model_desc;

/* Gaussian observations y = A x + eps.  HOST pointers, read during bta_create only.
 * Row i of A has a 1 at latent (time[i], var[i], node[i]) and cov[i][0..a/k) in fixed-effect columns
 * var[i]*(a/k) ...  (R11, R14). */
typedef struct {
  int64_t m;
  const int32_t* var;  /* [m] in [0,k) */
  const int32_t* node; /* [m] in [0,ns) */
  const int32_t* time; /* [m] in [0,nt) */
  const double* cov;   /* [m][a/k] */
  const double* y;     /* [m] */
} bta_obs;

/* DEVICE pointers to one BTA matrix (layouts above).  C may be NULL for BTA_PRIOR (C_i = 0). */
typedef struct {
  double* D;   /* [nt][b][b] */
  double* B;   /* [nt-1][b][b] */
  double* C;   /* [nt][a][b] */
  double* T;   /* [a][a] */
  double* rhs; /* [N] or NULL */
} bta_blocks;

/* Model setup: copies the observations to the device and reduces
 * them to theta-independent aggregates (counts, covariate sums, Z^T Z, A^T y) with device kernels in a
 * deterministic order.  `device` is the CUDA ordinal.  *out is NULL on failure. */
BTA_API int bta_create(bta_ctx** out, const bta_model_desc* desc, const bta_obs* obs, int device);
BTA_API int bta_destroy(bta_ctx* ctx);

/* Storage policy of inla_value_and_grad.
 *   BTA_STORE_FACTOR (default): the factor blocks X_t = L_Dt^-1 and L_Bt are kept for the backward sweep
 *     ((2nt-1) b^2 doubles per matrix, no recomputation).
 *   BTA_STORE_CARRY: the paper's carry-based reconstruction -- only the Schur-updated diagonal blocks
 *     D_t - S_{t-1} ("carries", nt b^2 doubles per matrix) and the O(a b) arrow rows / z_t are kept; the backward
 *     sweep rebuilds X_t (one more Cholesky + inverse) and L_Bt (B_t is re-assembled, one more product) per block.
 *   BTA_STORE_HOST: carry mode with the carries staged in page-locked HOST memory (§III-C c): each
 *     carry is copied out on a copy stream during the forward sweep and streamed back one block at a time, a few blocks
 *     ahead, during the backward sweep; the device keeps a ring of 4 diagonal-block slots per sub-chain, so the device
 *     workspace is O(b^2) whatever nt is.  Needs nt >= 3 (else it behaves as BTA_STORE_CARRY) and a host buffer of
 *     bta_host_bytes(ctx) bytes registered with bta_set_host_buffer before the next inla_value_and_grad.
 * Changes bta_workspace_bytes.  Returns BTA_ERR_ARG for an unknown mode. */
enum { BTA_STORE_FACTOR = 0, BTA_STORE_CARRY = 1, BTA_STORE_HOST = 2 };
BTA_API int bta_set_store_mode(bta_ctx* ctx, int mode);
BTA_API int bta_get_store_mode(const bta_ctx* ctx);
/* BTA_STORE_HOST: bytes of host staging memory needed (2 (nt-1) b^2 doubles), and its registration.  `host` is HOST
 * memory owned by the caller; it should be page-locked (cudaHostAlloc / torch pin_memory) -- pageable memory works but
 * the copies then do not overlap the sweeps.  It must stay valid until the mode is left or the ctx destroyed. */
BTA_API size_t bta_host_bytes(const bta_ctx* ctx);
BTA_API int bta_set_host_buffer(bta_ctx* ctx, void* host, size_t bytes);

/* Bytes of caller-provided device workspace needed by inla_value_and_grad (the largest user: both matrices'
 * blocks, per-chain temporaries).  bta_factor_logdet / bta_solve / bta_selinv need at most
 * bta_workspace_bytes_op(ctx) (three b x b temporaries + small vectors). */
BTA_API size_t bta_workspace_bytes(const bta_ctx* ctx);
BTA_API size_t bta_workspace_bytes_op(const bta_ctx* ctx);

/* Q_p(theta) or Q_c(theta) = Q_p + sum_v tau_v A_v^T A_v and r = sum_v tau_v A_v^T y_v as dense blocks
 * (Eq. 10 for k > 1 with the weights of R12).  theta: HOST, d doubles.  D is written
 * with its strict upper triangle ZERO (the lower triangle is authoritative everywhere in this library);
 * B, C, T in full.  out.rhs (if not NULL) receives r for BTA_COND, zeros for BTA_PRIOR. */
BTA_API int bta_assemble(bta_ctx* ctx, const double* theta, int which, bta_blocks out, void* stream);

/* Algorithm 1 (R8): block Cholesky Q = L L^T in place, and log det Q (HOST scalar).
 * The factor is kept in INVERSE-DIAGONAL FORM: on return
 *   D[t] = X_t = L_Dt^-1 (lower triangular, strict upper triangle zero),
 *   B[t] = L_Bt = B_t L_Dt^-T,   C[t] = L_Ct,   T = L_T (lower, strict upper zero),
 * and diagL (device, N doubles, may be NULL) receives diag(L_D1), ..., diag(L_Dnt), diag(L_T).
 * `which` = BTA_PRIOR skips the arrow (C ignored, T factored on its own).  Only the lower triangles of the
 * D[t] and T are read.  ws: device workspace (bta_workspace_bytes_op). */
BTA_API int bta_factor_logdet(bta_ctx* ctx, bta_blocks inout, int which, double* logdet, double* diagL, void* ws,
                      void* stream);

/* Both triangular sweeps L z = rhs, L^T x = z (Algorithm 1 line 5/11 and Eqs. 3-5) for
 * nrhs right-hand sides, in place: rhs_inout is DEVICE [nrhs][N].  L as left by bta_factor_logdet. */
BTA_API int bta_solve(bta_ctx* ctx, bta_blocks L, int which, double* rhs_inout, int nrhs, void* ws, void* stream);

/* BTA selected inversion (recurrences R10), in place over the factor left by
 * bta_factor_logdet: on return D[t] = Z_Dt = [Q^-1]_{tt} (both triangles), B[t] = Z_Bt = [Q^-1]_{t+1,t},
 * C[t] = Z_Ct = [Q^-1]_{T,t}, T = Z_T. */
BTA_API int bta_selinv(bta_ctx* ctx, bta_blocks inout, int which, void* ws, void* stream);

/* The hot path (PAPER.md:44 Eq. 1, :121 Eq. 6): f(theta) and grad f(theta).  theta HOST [d]; f HOST scalar;
 * grad HOST [d]; stage_ms HOST [BTA_NSTAGES] or NULL (CUDA-event times of the stages, see BTA_STAGE_*);
 * ws DEVICE, bta_workspace_bytes(ctx) bytes.  Runs assemble -> fused forward sweep -> fused backward sweep
 * (upper solve + selected inversion + trace contractions) on Q_c and on Q_p, then the scalar assembly. */
BTA_API int inla_value_and_grad(bta_ctx* ctx, const double* theta, double* f, double* grad, double* stage_ms, void* ws,
                        void* stream);

/* the objective alone (Eq. 1): assemble -> factor Q_c and Q_p -> solve ->
 * scalars; no selected inversion, no contractions.  One evaluation of the finite-difference baseline. */
BTA_API int inla_value(bta_ctx* ctx, const double* theta, double* f, void* ws, void* stream);

/* Central finite-difference gradient (Eq. 2; the DALIA baseline): 2d+1 calls of inla_value with
 * step h (the paper uses 1e-3).  f (may be NULL) receives f(theta), grad HOST [d].  Truncation error O(h^2). */
BTA_API int inla_fd_grad(bta_ctx* ctx, const double* theta, double h, double* f, double* grad, void* ws, void* stream);

/* posterior Hessian by central differences of the exact gradient (Eq. 13):
 * H[:, j] = (grad f(theta + h e_j) - grad f(theta - h e_j)) / (2h), 2d+1 calls of inla_value_and_grad (the centre
 * call returns f and grad, either may be NULL).  H HOST [d][d], as differenced (not symmetrised). */
BTA_API int inla_hessian(bta_ctx* ctx, const double* theta, double h, double* f, double* grad, double* H, void* ws,
                 void* stream);

/* the INLA mode search: maximise f(theta) (reading R1: Eq. 1 is a
 * log-posterior) by L-BFGS on -f with exact gradients from inla_value_and_grad and an Armijo backtracking line search;
 * host driver, no new kernels.  Stops when ||grad||_inf <= gtol or after max_iter iterations.  Outputs (HOST, any may
 * be NULL): theta_opt[d], f_opt, grad_opt[d], iters, evals (number of inla_value_and_grad calls). */
BTA_API int inla_optimize(bta_ctx* ctx, const double* theta0, int max_iter, double gtol, double* theta_opt, double* f_opt,
                  double* grad_opt, int* iters, int* evals, void* ws, void* stream);

/* Time-domain partitioning (§III-C a-b).  The nt time blocks are cut into P
 * contiguous partitions; partition 0 ends at one boundary block, every other partition has two; the interior blocks of
 * all partitions are eliminated concurrently (a partition p >= 1 carries a fill coupling to its top boundary), the
 * 2P-1 boundary blocks form a reduced BTA system that is factored and selectively inverted, and the interiors are
 * swept backwards concurrently, seeded by the reduced system's Sigma blocks.  Inside one GPU it is selected with
 * bta_set_option(ctx, BTA_OPT_PARTITIONS, P) (include/bta_diag.h) and inla_value_and_grad runs it whole.
 * bta_partition_plan returns the number of partitions actually used for a request of `partitions` (>= 2, <= 8,
 * clipped so that nt >= 2P-1) and their first / last time blocks (HOST arrays of >= 8 entries, may be NULL). */
BTA_API int bta_partition_plan(const bta_ctx* ctx, int partitions, int32_t* first, int32_t* last);

/* The same partitioning ACROSS ranks, one partition per rank (rank r of nranks owns partition r), with the paper's
 * communication pattern: no communication in Phase 1; ONE all-gather of the boundary data; every rank
 * solves the reduced system redundantly; ONE all-reduce of the partial sums.  The library does no communication
 * itself: the caller moves two device buffers between the three calls (the Python binding uses torch.distributed --
 * NCCL over NVLink on GPUs):
 *   1. inla_part_phase1: assembles and eliminates the interior of partition `rank` (both matrices) and packs its
 *      boundary data into `slab` (DEVICE, bta_part_slab_doubles(ctx) doubles): per matrix the updated boundary blocks
 *      D~(s_r), D~(e_r), the fill block Q~[e_r, s_r] and the tip accumulator, and for Q_c the stack rows [C~; r~] of
 *      both boundary blocks.  (The original couplings B_{e_p} are functions of theta and are assembled by every rank.)
 *      -> all-gather the slabs in rank order into `gathered` (nranks slabs).
 *   2. inla_part_phase2: unpacks all slabs, factors and selectively inverts the reduced system (2 nranks - 1 blocks),
 *      sweeps the interior of partition `rank` backwards and leaves the rank's per-block partial sums (traces,
 *      quadratic forms, log-determinant and residual partials; zeros for blocks of other ranks; the reduced system is
 *      counted by rank 0) in `partials` (DEVICE, caller-owned, bta_part_partial_doubles(ctx) doubles).
 *      -> all-reduce (sum) that buffer in place.
 *   3. inla_part_finish: f and grad f (HOST) from the summed partial sums -- identical on every rank.
 * Requires BTA_STORE_FACTOR, bta_set_option(ctx, BTA_OPT_PARTITIONS, nranks) (it sizes bta_workspace_bytes), the same
 * theta on every rank, and nt >= 2 nranks - 1.  x* from bta_last_intermediates is then valid only on the rank's own
 * and on the boundary blocks. */
BTA_API size_t bta_part_slab_doubles(const bta_ctx* ctx);
BTA_API int inla_part_phase1(bta_ctx* ctx, const double* theta, int rank, int nranks, double* slab, void* ws,
                             void* stream);
BTA_API size_t bta_part_partial_doubles(const bta_ctx* ctx);
BTA_API int inla_part_phase2(bta_ctx* ctx, int rank, int nranks, const double* gathered, double* partials, void* ws,
                             void* stream);
BTA_API int inla_part_finish(bta_ctx* ctx, const double* partials, double* f, double* grad, void* stream);

/* Allocation-free product for callers that cannot call cudaMalloc or provide scratch (code under CUDA-graph capture,
 * serving loops, harnesses that forbid allocation): the rows-times-block product of the upper solve and of the arrow
 * recurrences (Eqs. 3-5; R10),
 *     out[p][j] = alpha * sum_{k >= kbeg(j)} R[p][k] * M[k][j] + beta * in[p][j],   kbeg(j) = tri ? j : 0,
 * P <= 9 rows R (ldr) against a K x J block M (ldm; tri = 1: M lower triangular), all DEVICE pointers, row-major FP64;
 * `in` may be NULL when beta = 0 and may alias `out`.  The kernel's partial-sum scratch (ceil(K/128) * P * J doubles)
 * is a file-scope device array of BTA_NOALLOC_MAX_PART doubles (9.4 MB: enough for P = 9, K = J = 4096) that every
 * GPU loading the library holds until exit; larger products are rejected with BTA_ERR_ARG and a message.  The call
 * allocates nothing (no cudaMalloc / cudaFree, no allocating library routine), launches on `stream` on the CURRENT
 * device and does not synchronise.  All calls on one device share the array, which keeps the last call's contents
 * (every entry read is written first by the same call, so nothing needs clearing): calls that overlap on the GPU
 * race -- issue them on one stream or order them with events. */
#define BTA_NOALLOC_MAX_PART (32 * 9 * 4096)
BTA_API int bta_rows_times_block_noalloc(int P, int K, int J, const double* R, int ldr, const double* M, int ldm, int tri,
                                         double alpha, double beta, const double* in, int ldin, double* out, int ldo,
                                         void* stream);

enum {
  BTA_STAGE_ASSEMBLE = 0,
  BTA_STAGE_FWD_QC = 1,
  BTA_STAGE_BWD_QC = 2,
  BTA_STAGE_FWD_QP = 3,
  BTA_STAGE_BWD_QP = 4,
  BTA_STAGE_SCALARS = 5,
  BTA_STAGE_TOTAL = 6,
  BTA_NSTAGES = 7
};

/* Intermediates of the last inla_value_and_grad (HOST outputs; any pointer may be NULL):
 * ld[2] = {log det Q_p, log det Q_c}; x DEVICE->HOST copy of x* [N]; parts[3*d] = Phase A, B, C per
 * hyperparameter (Eq. 6 terms before the -1/2, -1/2, +1/2 factors); rss[k] = ||y_v - A_v x*||^2;
 * quad = x*^T Q_p x*; ZT[a*a] = Z_T = [Q_c^-1]_{TT}. */
BTA_API int bta_last_intermediates(bta_ctx* ctx, double* ld, double* x, double* parts, double* rss, double* quad,
                           double* ZT);

BTA_API int32_t bta_num_hyper(const bta_ctx* ctx);  /* d */
BTA_API int64_t bta_latent_size(const bta_ctx* ctx); /* N */
BTA_API int64_t bta_last_pivot(const bta_ctx* ctx);  /* 1-based global row of the first non-positive pivot, 0 if none */
BTA_API int64_t bta_kernel_launches(const bta_ctx* ctx); /* kernels launched by this ctx so far */
BTA_API const char* bta_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* BTA_H_ */
