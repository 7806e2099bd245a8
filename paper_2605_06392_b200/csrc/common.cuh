// Shared declarations of the sm_100a BTA / INLA library (internal; the public boundary is include/bta.h).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "../../include/bta.h"
#include "../../include/bta_diag.h"

#define BTA_CUDA_OK(call)                                                              \
  do {                                                                                 \
    cudaError_t e_ = (call);                                                           \
    if (e_ != cudaSuccess) {                                                           \
      bta_set_error_cuda(e_, #call, __FILE__, __LINE__);                               \
      return BTA_ERR_CUDA;                                                             \
    }                                                                                  \
  } while (0)

void bta_set_error_cuda(cudaError_t e, const char* what, const char* file, int line);
void bta_set_error(const char* msg);

// Every entry point runs on the ctx's device and restores the caller's current device on return.
struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(int device) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    if (prev != device) cudaSetDevice(device);
    else prev = -1;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is a per-device setting: opt in once per (kernel, device).
// `done` is one bit per device ordinal, owned by the caller (one static per kernel instantiation).
template <class K>
cudaError_t optin_smem(K kern, int bytes, unsigned long long* done_bits) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const unsigned long long bit = 1ull << (dev & 63);
  if (__atomic_load_n(done_bits, __ATOMIC_ACQUIRE) & bit) return cudaSuccess;
  e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e != cudaSuccess) return e;
  __atomic_fetch_or(done_bits, bit, __ATOMIC_RELEASE);
  return cudaSuccess;
}

// Per-kernel-class timing (ktime.cu; bta_diag.h: BTA_KC_*): a scope object around each kernel launch.
extern bool g_ktime_on;
struct KTimeScope {
  long long idx;
  cudaStream_t stream;
  KTimeScope(int cls, cudaStream_t st, double flop, double bytes);
  ~KTimeScope();
  KTimeScope(const KTimeScope&) = delete;
  KTimeScope& operator=(const KTimeScope&) = delete;
};

// ------------------------------------------------------------------------------------------------
// FP64 DMMA GEMM  (gemm.cu):  C = alpha * op(A) op(B) + beta * C, row-major, optionally batched
// ------------------------------------------------------------------------------------------------
enum : int {
  GEMM_NN = 0,  // A [M][K], B [K][N]
  GEMM_NT = 1,  // A [M][K], B [N][K]
  GEMM_TN = 2,  // A [K][M], B [K][N]
};
// Restriction of the contraction range per output tile (triangular operands; tile-aligned).
enum : int {
  KLO_ZERO = 0,  // k >= 0
  KLO_N0 = 1,    // k >= first column of the tile   (lower-triangular B in NN: B[k][n] = 0 for k < n)
  KLO_M0 = 2,    // k >= first row of the tile      (X^T X lower part: k >= max(m, n) = m)
};
enum : int {
  KHI_K = 0,      // k < K
  KHI_NEND = 1,   // k < last column of the tile + 1 (lower-triangular B in NT: B[n][k] = 0 for k > n)
  KHI_MEND = 2,   // k < last row of the tile + 1    (lower-triangular A in NN: A[m][k] = 0 for k > m)
};
enum : int {
  OUT_FULL = 0,
  OUT_LOWER = 1,         // write only elements with m >= n (tiles above the diagonal are skipped)
  OUT_LOWER_MIRROR = 2,  // compute m >= n, write C[m][n] and C[n][m]
};

struct GemmSub {  // one problem of a batched launch: element offsets from the base pointers
  long long offA, offB, offC;
  int M, N, K, pad;
};

struct GemmArgs {
  const double* A;
  const double* B;
  double* C;
  int M, N, K;
  int lda, ldb, ldc;
  double alpha, beta;
  int mode, klo, khi, out;
  const GemmSub* subs;  // device array (nsub problems; M,N,K above = maxima for the grid) or nullptr
  int nsub;
  int group;            // tile-order grouping (set by launch_gemm): slow tile rows swept together, <= 1 = off
};

extern long long g_tile_thresh;
extern int g_tile_waves;
// Programmatic dependent launch for the latency-bound kernels (POTRF leaves, 32x32-tile GEMMs): the kernel is launched
// with cudaLaunchAttributeProgrammaticStreamSerialization, starts while its predecessor in the stream drains, and waits
// at `griddepcontrol.wait` before touching memory.  BTA_OPT_PDL (process-global): 0 off, 1 both kernel classes, 2 the
// GEMMs only, 3 the leaves only (default: early-resident GEMM CTAs cost more SM slots than their start-up saves).
extern int g_pdl;
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <class... KArgs, class... Args>
cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}
cudaError_t launch_gemm(const GemmArgs& g, cudaStream_t st);
bool gemm_uses_small_tiles(const GemmArgs& g);  // the 64x64-tile configuration (few CTAs)

// ------------------------------------------------------------------------------------------------
// Leaf / tip kernels (diag.cu)
// ------------------------------------------------------------------------------------------------
// leaf.cu: POTRF + TRTRI of one n x n (n <= leaf_max_n() = 144) diagonal tile in one CTA (16-wide panels, DMMA updates)
int leaf_max_n();
cudaError_t launch_potrf_inv_blocked(double* A, int ld, int n, double* diagL, long long grow0,
                                     unsigned long long* pivot_flag, cudaStream_t st);
cudaError_t launch_tip(const double* Tt, int a, int nr, int do_chol, double* LT, double* zT, double* xT, double* ZT,
                       double* diagL, long long grow0, unsigned long long* pivot_flag, cudaStream_t st);
cudaError_t launch_zero_upper(double* A, int ld, int n, cudaStream_t st);
cudaError_t launch_tip_inverse(const double* LT, int a, double* ZT, cudaStream_t st);

// ------------------------------------------------------------------------------------------------
// Skinny (arrow / vector) kernels (skinny.cu)
// ------------------------------------------------------------------------------------------------
cudaError_t launch_skinny_nt(int P, int J, int K, const double* R, int ldr, const double* M, int ldm, int tri,
                             double alpha, double beta, const double* in, int ldin, double* out, int ldo,
                             cudaStream_t st);
size_t skinny_nn_part_doubles(int P, int K, int J);
cudaError_t launch_skinny_nn(int P, int K, int J, const double* R, int ldr, const double* M, int ldm, int tri,
                             double alpha, double beta, const double* in, int ldin, double* out, int ldo,
                             double* part, cudaStream_t st);
cudaError_t launch_small_nt(int PU, int PV, int K, const double* U, int ldu, const double* V, int ldv, double alpha,
                            double* Tt, int ldt, cudaStream_t st);
// Y[r][j] = beta * In[r][j] + alpha * sum_q S[r][q] * E[q][j]   (S: R x Q, lds; E: Q x J)
cudaError_t launch_small_left_mul(int R, int Q, int J, const double* S, int lds, const double* E, int lde,
                                  double alpha, double beta, const double* In, int ldin, double* Y, int ldy,
                                  cudaStream_t st);

// ------------------------------------------------------------------------------------------------
// Model context, theta-derived parameters (model.cu), assembly (assemble.cu), contractions (contract.cu)
// ------------------------------------------------------------------------------------------------
constexpr int KMAX = 4;    // response variables
constexpr int AMAX = 8;    // arrow width (skinny kernels hold a+1 <= 9 rows)
constexpr int DMAX = 3 * KMAX + KMAX * (KMAX - 1) / 2 + KMAX;

struct DevParams {          // lives in device memory; written by theta_prep_kernel
  double theta[DMAX];
  double E[KMAX][3];        // exp(theta_{m,c})
  double Lam[KMAX][KMAX];   // unit lower-triangular coupling (R12)
  double tau[KMAX];         // noise precisions
  double W[3][KMAX][KMAX];  // W_c[i][j] = sum_m E[m][c] Lam[m][i] Lam[m][j]  (Eq. 10)
};

struct ModelDims {
  int nt, g, ns, k, a, apr, b, d;
  long long N;
  double h, fixed_prec;
};

constexpr int BTA_NSW = 256;

// Run-time options (include/bta_diag.h: bta_set_option; defaults = the measured best, or BTA_* environment variables
// read once in bta_create).
struct Options {
  int twist = 1;      // two-way elimination (four chains); 0: one chain per matrix
  int lanes = 1;      // high-priority companion streams for the small kernels (2: forward sweeps only)
  int split = 1;      // coupled forward step for b <= 1024
  int graph = -1;     // CUDA-graph replay from the second call on: -1 = by size (b <= 1024), 0 off, 1 on
  int serial = 0;     // both matrices on one stream, single chain (exclusive per-stage times)
  int pipeline = 1;   // forward sweeps: start the next block's factorisation under the tail of this block's products
  int rows = 1;       // arrow / rhs rows and trace contractions on a third stream per chain (factor mode)
  int partitions = 0; // >= 2: time-domain partitioning with that many partitions and a reduced system (partition.cu)
};

struct bta_ctx {
  ModelDims md;
  Options opt;
  int device;
  long long m;
  // observations on the device
  int *o_var, *o_node, *o_time;
  double *o_cov, *o_y;
  // theta-independent aggregates
  double *cnt, *zsum, *ZZ, *ysum, *zy, *yy, *mv;  // [nt][b], [nt][a][b], [k][a][a], [nt][b], [k][a], [k], [k]
  DevParams* P;
  double* theta_dev;                 // staging for H2D of theta
  unsigned long long* pivot_flag;    // device; ~0ull = none
  double* small;                     // device scratch for tips, partial sums, outputs (carved in model.cu)
  size_t small_doubles;
  double* host_pinned;               // pinned host staging (theta in, f/grad/intermediates out)
  cudaStream_t s_side;               // second chain's stream
  cudaStream_t s_main;               // graph mode: the captured/replayed stream (the caller's may be stream 0)
  cudaGraphExec_t graph_exec[2];     // cached replay of one whole gradient [0] / value-only pass [1], or nullptr
  void* graph_ws[2];                 // workspace pointer the cached graph was captured with
  long long graph_launches[2];       // kernels inside the cached graph
  long long grad_calls;
  int store_mode;                    // BTA_STORE_FACTOR / BTA_STORE_CARRY
  cudaStream_t s_aux[2];             // two-way elimination: the down chains of Q_c and Q_p
  cudaEvent_t ev[32];
  cudaStream_t s_hi[4];              // high-priority companions of the four chains (small kernels)
  cudaStream_t s_x[4];               // side streams of the four chains (off-chain work of the forward steps)
  double* host_buf;                  // BTA_STORE_HOST: caller-owned page-locked staging memory for the carries
  size_t host_bytes;
  cudaStream_t s_copy[4];            // its copy streams (one per sub-chain) and ring-slot events
  cudaEvent_t ev_ring[4][8];
  cudaEvent_t ev_pipe[20][17];       // per chain (sweep.h: Chain::pipe_ev): forward pipelining [0..2], trace parity [3..4];
                                     // backward work running ahead on the solve stream, by step parity: arrow products
                                     // E, Z_T E ready [5..6] / consumed [7..8], G and X^T X ready [9..10], G consumed
                                     // [11..12], Z_D buffer read by the next step's Z_B product [13..14]
  cudaStream_t s_r[4];               // rows streams of the four chains (sweep.h: Chain::rs)
  cudaStream_t s_g[4];               // G / X^T X streams of the four chains in the backward sweep (sweep.h: Chain::gs)
  cudaStream_t s_part[2][8], s_part_hi[2][8], s_part_x[2][8], s_part_r[2][8];  // partition.cu: per (matrix, partition)
  cudaEvent_t ev_sw[256];            // lane-switch events, used round-robin
  unsigned ev_sw_next;
  long long launches;
  long long last_pivot;
  // last intermediates (host)
  double last_ld[2], last_quad;
  std::vector<double> last_parts, last_rss;
  double* x_keep;                    // library-owned copy of x* of the last gradient (N doubles)
  bool have_x;
  // BTA_TRACE=<file>: phase marks of the sweeps (diagnostic timeline; events are created on demand)
  struct TraceRec { cudaEvent_t e; int chain, t, tag; };
  std::vector<TraceRec> trace;
  bool trace_on;
};
inline void trace_mark(bta_ctx* c, cudaStream_t st, int chain, int t, int tag) {
  if (!c->trace_on) return;
  cudaEvent_t e;
  cudaEventCreate(&e);
  cudaEventRecord(e, st);
  c->trace.push_back({e, chain, t, tag});
}

#define BTA_COUNT(ctx) ((ctx)->launches++)

// assemble.cu
cudaError_t launch_theta_prep(bta_ctx* c, cudaStream_t st);
// Writes D (strict upper zero), B, the arrow rows C (block stride c_stride, row stride b), T and the rhs
// (time block t at rhs + t * rhs_stride; tip at rhs_tip).  Any of B, C, T, rhs may be NULL.
cudaError_t launch_assemble(bta_ctx* c, int which, double* D, long long d_stride, double* B, long long b_stride,
                            double* C, long long c_stride, double* T, int ldt, double* rhs, long long rhs_stride,
                            double* rhs_tip, int rhs_tip_stride, cudaStream_t st);
cudaError_t run_setup_aggregates(bta_ctx* c, cudaStream_t st);
// One sub-diagonal block B_t (kind 1) or diagonal block D_t (kind 0) into `out` (b x b).
cudaError_t launch_assemble_block(bta_ctx* c, int which, int kind, int t, int transpose, double* out,
                                  cudaStream_t st);
// `count` blocks t0, t0+tdir, ... of kind 0 (D) / 1 (B; transposed if `transpose`) into out + z * stride.
cudaError_t launch_assemble_seq(bta_ctx* c, int which, int kind, int t0, int tdir, int count, int transpose,
                                double* out, long long stride, cudaStream_t st);

// contract.cu -- layout of the small device scratch (offsets in doubles into bta_ctx::small)
struct SmallLayout {
  int nx;                       // CTAs along the node axis of the stencil kernels = ceil(ns / 256)
  size_t trc[2];                // [chain][nt][2][k][k][nx][3]   traces <Z^(ij), K_c> per block, per CTA
  size_t qd;                    // [nt][2][k][k][nx][3]          x^(i)T K_c x^(j)
  size_t noise;                 // [nt][k][nx]
  size_t ldpart[2];             // [64]
  size_t rsspart;               // [256][k]
  size_t Tt[2], LT[2], zT[2], xT[2], ZT[2];   // tips per chain
  size_t out;                   // f, grad[d], ld[2], parts[3d], rss[k], quad
  size_t total;
};
SmallLayout small_layout(const ModelDims& md);
enum { CH_PRIOR = 0, CH_COND = 1 };

cudaError_t launch_trace_stencil(bta_ctx* c, int chain, int t, int kind, const double* Z, int ld, cudaStream_t st);
cudaError_t launch_noise_trace(bta_ctx* c, int t, const double* ZD, int ld, const double* ZC, int ldzc,
                               cudaStream_t st);
cudaError_t launch_quad_stencil(bta_ctx* c, const double* x, cudaStream_t st);
// ... restricted to the time blocks [t_lo, t_hi] (a rank's partition): the other blocks' partial sums are written as 0
cudaError_t launch_quad_stencil(bta_ctx* c, const double* x, int t_lo, int t_hi, cudaStream_t st);
cudaError_t launch_residual(bta_ctx* c, const double* x, int t_lo, int t_hi, cudaStream_t st);
cudaError_t launch_logdet_partial(bta_ctx* c, int chain, const double* dvec, cudaStream_t st);
cudaError_t launch_residual(bta_ctx* c, const double* x, cudaStream_t st);
cudaError_t launch_scalars(bta_ctx* c, cudaStream_t st);
cudaError_t launch_logdet_final(bta_ctx* c, int chain, double* out, cudaStream_t st);
