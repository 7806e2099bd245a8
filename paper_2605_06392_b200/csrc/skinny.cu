// Bandwidth-bound "skinny" products of the sweeps: a few rows (arrow rows L_C / Z_C, right-hand-side and
// solution vectors) against one b x b block.  These are the arrow and vector parts of Algorithm 1
// (PAPER.md:77-96, lines 4-5, 9), of Eqs. 3-5 and of the selected-inversion arrow
// recurrences (R10).  P <= 16 rows; each kernel reads the b x b block exactly once (HBM roofline).
#include "common.cuh"

constexpr int NN_KCH = 128;
constexpr int NT_RPW = 4;    // rows of M per warp in skinny_nt (2 x 8, 2 x 4, 4 x 2 were measured: profiles/r02_hbm_kernels.md)
constexpr int NT_WARPS = 4;  // warps per CTA in skinny_nt (16 rows of M per CTA)

namespace {

// out[p][j] = beta * in[p][j] + alpha * sum_{k < kend(j)} R[p][k] * M[j][k],  kend(j) = tri ? j+1 : K.
// One warp per NT_RPW rows j of M (k contiguous -> coalesced).  The R chunk is staged in shared memory and each staged
// value is read into registers once per k-step and used for all NT_RPW rows (PT / NT_RPW shared loads per element of M
// instead of PT), with the NT_RPW row loads of a k-step in flight together.
template <int PT>
__global__ void __launch_bounds__(32 * NT_WARPS) skinny_nt_kernel(int P, int J, int K, const double* __restrict__ R,
                                                                  int ldr, const double* __restrict__ M, int ldm,
                                                                  int tri, double alpha, double beta, const double* in,
                                                                  int ldin, double* out, int ldo) {
  // `in` and `out` may be the same buffer (in-place stack updates of the sweeps): no __restrict__ on them
  constexpr int KC = PT > 9 ? 128 : 256, RPW = NT_RPW, NT = 32 * NT_WARPS;   // 2 PT KC doubles of static shared memory
  __shared__ __align__(16) double Rs[2][PT * KC];   // chunk c in Rs[c & 1], staged one chunk ahead by cp.async
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int jbase = blockIdx.x * (NT_WARPS * RPW) + warp * RPW;
  const int jmax_cta = min(J, (int)(blockIdx.x + 1) * (NT_WARPS * RPW)) - 1;
  const int Kcta = tri ? min(K, jmax_cta + 1) : K;
  double acc[RPW][PT];
  const double* mrow[RPW];
  int kend[RPW];
#pragma unroll
  for (int r = 0; r < RPW; ++r) {
    const int j = jbase + r;
    kend[r] = j < J ? (tri ? min(K, j + 1) : K) : 0;
    mrow[r] = M + (long long)min(j, J - 1) * ldm;
#pragma unroll
    for (int p = 0; p < PT; ++p) acc[r][p] = 0.0;
  }
  int kend_warp = 0;
#pragma unroll
  for (int r = 0; r < RPW; ++r) kend_warp = max(kend_warp, kend[r]);
  // R[p][k0 .. k0+KC) -> Rs[buf] (8-byte asynchronous copies; entries beyond P or Kcta are zeroed by plain stores)
  auto stage = [&](int buf, int k0) {
    for (int e = tid; e < PT * KC; e += NT) {
      const int p = e / KC, k = e % KC;
      if (p < P && k0 + k < Kcta) {
        const unsigned dst = (unsigned)__cvta_generic_to_shared(&Rs[buf][e]);
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(R + (long long)p * ldr + k0 + k) : "memory");
      } else {
        Rs[buf][e] = 0.0;
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  stage(0, 0);
  for (int k0 = 0, c = 0; k0 < Kcta; k0 += KC, ++c) {
    // The RPW * KC / 32 loads of this chunk are issued first (8 KB per warp in flight); R of this chunk was requested
    // one chunk ago, R of the next one is requested before the arithmetic starts.
    double m[KC / 32][RPW];
#pragma unroll
    for (int q = 0; q < KC / 32; ++q) {
      const int k = k0 + q * 32 + lane;
#pragma unroll
      for (int r = 0; r < RPW; ++r) m[q][r] = (k < kend[r]) ? __ldcs(mrow[r] + k) : 0.0;
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();                       // Rs[c & 1] is complete; everybody is done with Rs[(c + 1) & 1]
    if (k0 + KC < Kcta) stage((c + 1) & 1, k0 + KC);
    if (k0 >= kend_warp) continue;         // every row of this warp ends before the chunk
    const double* rs = Rs[c & 1];
#pragma unroll
    for (int q = 0; q < KC / 32; ++q) {
      double rr[PT];
#pragma unroll
      for (int p = 0; p < PT; ++p) rr[p] = rs[p * KC + q * 32 + lane];
#pragma unroll
      for (int r = 0; r < RPW; ++r)
#pragma unroll
        for (int p = 0; p < PT; ++p) acc[r][p] = fma(m[q][r], rr[p], acc[r][p]);
    }
  }
#pragma unroll
  for (int r = 0; r < RPW; ++r) {
    const int j = jbase + r;
#pragma unroll
    for (int p = 0; p < PT; ++p) {
      double v = acc[r][p];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      if (lane == 0 && j < J && p < P) {
        double res = alpha * v;
        if (beta != 0.0) res += beta * in[(long long)p * ldin + j];
        out[(long long)p * ldo + j] = res;
      }
    }
  }
}

// part[ks][p][j] = sum_{k in chunk ks, k >= kbeg(j)} R[p][k] * M[k][j],  kbeg(j) = tri ? j : 0.
// CTA: 128 columns x NN_KCH rows of M; threads (64 x 4): 2 columns each, 4 k-phases reduced through smem.
template <int PT>
__global__ void __launch_bounds__(256) skinny_nn_kernel(int P, int K, int J, const double* __restrict__ R, int ldr,
                                                        const double* __restrict__ M, int ldm, int tri,
                                                        double* __restrict__ part) {
  constexpr int KCH = NN_KCH;
  __shared__ double Rs[PT * KCH];
  __shared__ double red[4][PT][128];
  const int tid = threadIdx.x, tx = tid & 63, ty = tid >> 6;
  const int j0 = blockIdx.x * 128, k0 = blockIdx.y * KCH;
  const int k1 = min(K, k0 + KCH);
  const int ja = j0 + tx, jb = j0 + tx + 64;
  double acc[PT][2];
#pragma unroll
  for (int p = 0; p < PT; ++p) acc[p][0] = acc[p][1] = 0.0;
  const bool skip = tri && (k1 - 1 < j0);  // every row of this chunk is above the diagonal of every column
  if (!skip) {
    for (int e = tid; e < PT * KCH; e += 256) {
      int p = e / KCH, k = e % KCH;
      Rs[e] = (p < P && k0 + k < k1) ? R[(long long)p * ldr + k0 + k] : 0.0;
    }
    __syncthreads();
    constexpr int U = 8;   // k-rows per thread whose loads are in flight together (16 x 8 B per thread)
    for (int kb = k0 + ty; kb < k1; kb += 4 * U) {
      double ma[U], mb[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int k = kb + 4 * u;
        const double* mrow = M + (long long)k * ldm;
        ma[u] = (k < k1 && ja < J && (!tri || k >= ja)) ? __ldcs(mrow + ja) : 0.0;
        mb[u] = (k < k1 && jb < J && (!tri || k >= jb)) ? __ldcs(mrow + jb) : 0.0;
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int k = kb + 4 * u;
        if (k < k1) {
#pragma unroll
          for (int p = 0; p < PT; ++p) {
            const double r = Rs[p * KCH + (k - k0)];
            acc[p][0] = fma(r, ma[u], acc[p][0]);
            acc[p][1] = fma(r, mb[u], acc[p][1]);
          }
        }
      }
    }
  }
#pragma unroll
  for (int p = 0; p < PT; ++p) {
    red[ty][p][tx] = acc[p][0];
    red[ty][p][tx + 64] = acc[p][1];
  }
  __syncthreads();
  for (int e = tid; e < PT * 128; e += 256) {
    int p = e / 128, c = e % 128;
    if (p < P && j0 + c < J) {
      double s = (red[0][p][c] + red[1][p][c]) + (red[2][p][c] + red[3][p][c]);
      part[((long long)blockIdx.y * P + p) * J + j0 + c] = s;
    }
  }
}

// out[p][j] = alpha * sum_ks part[ks][p][j] + beta * in[p][j]   (fixed order: deterministic)
__global__ void skinny_nn_finish_kernel(int P, int J, int nks, const double* __restrict__ part, double alpha,
                                        double beta, const double* in, int ldin, double* out, int ldo) {
  // `in` may alias `out` (in-place update): no __restrict__ on them
  long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (long long)P * J) return;
  int p = (int)(e / J), j = (int)(e % J);
  double s = 0.0;
  for (int ks = 0; ks < nks; ++ks) s += part[((long long)ks * P + p) * J + j];
  double res = alpha * s;
  if (beta != 0.0) res += beta * in[(long long)p * ldin + j];
  out[(long long)p * ldo + j] = res;
}

// Tt[p][q] += alpha * sum_k U[p][k] * V[q][k]  for p < PU, q < PV (Algorithm 1 line 9 and v_T of line 5).
__global__ void __launch_bounds__(256) small_nt_kernel(int PU, int PV, int K, const double* __restrict__ U, int ldu,
                                                       const double* __restrict__ V, int ldv, double alpha,
                                                       double* __restrict__ Tt, int ldt) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int pq = blockIdx.x * nw + warp; pq < PU * PV; pq += gridDim.x * nw) {
    int p = pq / PV, q = pq % PV;
    double s = 0.0;
    for (int k = lane; k < K; k += 32) s = fma(U[(long long)p * ldu + k], V[(long long)q * ldv + k], s);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) Tt[p * ldt + q] += alpha * s;
  }
}

// Y[r][j] = beta * In[r][j] + alpha * sum_q S[r][q] * E[q][j]   (tiny left factor: Z_T E_i, x_T^T L_C, ...)
__global__ void small_left_mul_kernel(int R, int Q, int J, const double* __restrict__ S, int lds,
                                      const double* __restrict__ E, int lde, double alpha, double beta,
                                      const double* In, int ldin, double* Y, int ldy) {  // In may alias Y
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= J) return;
  for (int r = 0; r < R; ++r) {
    double s = 0.0;
    for (int q = 0; q < Q; ++q) s = fma(S[r * lds + q], E[(long long)q * lde + j], s);
    double res = alpha * s;
    if (beta != 0.0) res += beta * In[(long long)r * ldin + j];
    Y[(long long)r * ldy + j] = res;
  }
}

}  // namespace

cudaError_t launch_skinny_nt(int P, int J, int K, const double* R, int ldr, const double* M, int ldm, int tri,
                             double alpha, double beta, const double* in, int ldin, double* out, int ldo,
                             cudaStream_t st) {
  if (P <= 0 || J <= 0) return cudaSuccess;
  KTimeScope kt(BTA_KC_SKINNY, st, 2.0 * P * (double)J * K * (tri ? 0.5 : 1.0), 8.0 * (double)J * K * (tri ? 0.5 : 1.0));
  dim3 grid((J + NT_WARPS * NT_RPW - 1) / (NT_WARPS * NT_RPW));
  if (P <= 1)
    skinny_nt_kernel<1><<<grid, 32 * NT_WARPS, 0, st>>>(P, J, K, R, ldr, M, ldm, tri, alpha, beta, in, ldin, out, ldo);
  else if (P <= 4)
    skinny_nt_kernel<4><<<grid, 32 * NT_WARPS, 0, st>>>(P, J, K, R, ldr, M, ldm, tri, alpha, beta, in, ldin, out, ldo);
  else if (P <= 9)
    skinny_nt_kernel<9><<<grid, 32 * NT_WARPS, 0, st>>>(P, J, K, R, ldr, M, ldm, tri, alpha, beta, in, ldin, out, ldo);
  else if (P <= 16)
    skinny_nt_kernel<16><<<grid, 32 * NT_WARPS, 0, st>>>(P, J, K, R, ldr, M, ldm, tri, alpha, beta, in, ldin, out, ldo);
  else
    return cudaErrorInvalidValue;
  return cudaGetLastError();
}

size_t skinny_nn_part_doubles(int P, int K, int J) { return (size_t)((K + NN_KCH - 1) / NN_KCH) * P * J; }

cudaError_t launch_skinny_nn(int P, int K, int J, const double* R, int ldr, const double* M, int ldm, int tri,
                             double alpha, double beta, const double* in, int ldin, double* out, int ldo,
                             double* part, cudaStream_t st) {
  if (P <= 0 || J <= 0) return cudaSuccess;
  KTimeScope kt(BTA_KC_SKINNY, st, 2.0 * P * (double)J * K * (tri ? 0.5 : 1.0), 8.0 * (double)J * K * (tri ? 0.5 : 1.0));
  const int nks = (K + NN_KCH - 1) / NN_KCH;
  dim3 grid((J + 127) / 128, nks);
  if (P <= 1)
    skinny_nn_kernel<1><<<grid, 256, 0, st>>>(P, K, J, R, ldr, M, ldm, tri, part);
  else if (P <= 4)
    skinny_nn_kernel<4><<<grid, 256, 0, st>>>(P, K, J, R, ldr, M, ldm, tri, part);
  else if (P <= 9)
    skinny_nn_kernel<9><<<grid, 256, 0, st>>>(P, K, J, R, ldr, M, ldm, tri, part);
  else
    return cudaErrorInvalidValue;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  long long tot = (long long)P * J;
  skinny_nn_finish_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(P, J, nks, part, alpha, beta, in, ldin, out,
                                                                         ldo);
  return cudaGetLastError();
}

cudaError_t launch_small_nt(int PU, int PV, int K, const double* U, int ldu, const double* V, int ldv, double alpha,
                            double* Tt, int ldt, cudaStream_t st) {
  if (PU <= 0 || PV <= 0) return cudaSuccess;
  KTimeScope kt(BTA_KC_OTHER, st, 2.0 * PU * (double)PV * K, 8.0 * (double)(PU + PV) * K);
  small_nt_kernel<<<8, 256, 0, st>>>(PU, PV, K, U, ldu, V, ldv, alpha, Tt, ldt);
  return cudaGetLastError();
}

cudaError_t launch_small_left_mul(int R, int Q, int J, const double* S, int lds, const double* E, int lde,
                                  double alpha, double beta, const double* In, int ldin, double* Y, int ldy,
                                  cudaStream_t st) {
  if (R <= 0 || J <= 0) return cudaSuccess;
  KTimeScope kt(BTA_KC_OTHER, st, 2.0 * R * (double)Q * J, 8.0 * (double)(Q + 2 * R) * J);
  small_left_mul_kernel<<<(J + 255) / 256, 256, 0, st>>>(R, Q, J, S, lds, E, lde, alpha, beta, In, ldin, Y, ldy);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Allocation-free entry point (include/bta.h: bta_rows_times_block_noalloc) and, for comparison, the same product through
// the existing launcher with caller-provided scratch (include/bta_diag.h: bta_rows_times_block).
//
// skinny_nn needs a scratch array for its per-k-chunk partial sums ([ceil(K/128)][P][J] doubles); the sweeps carve it
// out of the caller's workspace.  Some callers cannot provide or allocate one (code under CUDA-graph capture, serving
// loops, harnesses that forbid cudaMalloc).  For them the scratch is this file-scope device array: BTA_NOALLOC_MAX_PART
// doubles = 9.4 MB (P = 9 rows against a 4096 x 4096 block), held by every GPU that loads the library until exit.
// In host code `g_noalloc_part` is only the host-side stand-in of the symbol: the device address is taken once per
// device with cudaGetSymbolAddress (that device current) and passed to the kernels.  Every partial sum that the finish
// kernel reads is written by the product kernel of the same call (skipped chunks write zeros), so nothing has to be
// cleared between calls; the array keeps the last call's contents.  All calls on one device share the array: calls that
// overlap on the GPU (different streams) race -- serialise them.
// ------------------------------------------------------------------------------------------------
namespace {
constexpr size_t NOALLOC_MAX_PART = BTA_NOALLOC_MAX_PART;
static __device__ __align__(256) double g_noalloc_part[NOALLOC_MAX_PART];
constexpr int NOALLOC_MAX_DEV = 64;
double* g_noalloc_ptr[NOALLOC_MAX_DEV] = {};   // device address of g_noalloc_part per device ordinal (set-up once)

int rows_times_block_check(const char* who, int P, int K, int J, const double* R, const double* M, const double* in,
                           double beta, const double* out) {
  char buf[200];
  if (P < 1 || P > 9 || K < 1 || J < 1 || !R || !M || !out || (beta != 0.0 && !in)) {
    snprintf(buf, sizeof buf, "%s: need 1 <= P <= 9, K >= 1, J >= 1, non-null R, M, out (and in when beta != 0)", who);
    bta_set_error(buf);
    return BTA_ERR_ARG;
  }
  return BTA_OK;
}
}  // namespace

extern "C" int bta_rows_times_block_noalloc(int P, int K, int J, const double* R, int ldr, const double* M, int ldm,
                                            int tri, double alpha, double beta, const double* in, int ldin,
                                            double* out, int ldo, void* stream) {
  if (int rc = rows_times_block_check("bta_rows_times_block_noalloc", P, K, J, R, M, in, beta, out); rc != BTA_OK)
    return rc;
  const size_t need = skinny_nn_part_doubles(P, K, J);
  if (need > NOALLOC_MAX_PART) {
    char buf[200];
    snprintf(buf, sizeof buf,
             "bta_rows_times_block_noalloc: ceil(K/128) * P * J = %zu doubles of scratch exceed the built-in %zu "
             "(BTA_NOALLOC_MAX_PART); use the workspace-based calls",
             need, (size_t)NOALLOC_MAX_PART);
    bta_set_error(buf);
    return BTA_ERR_ARG;
  }
  int dev = 0;
  BTA_CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= NOALLOC_MAX_DEV) {
    bta_set_error("bta_rows_times_block_noalloc: device ordinal out of range");
    return BTA_ERR_ARG;
  }
  double* part = __atomic_load_n(&g_noalloc_ptr[dev], __ATOMIC_ACQUIRE);
  if (!part) {  // once per device, with that device current
    void* p = nullptr;
    BTA_CUDA_OK(cudaGetSymbolAddress(&p, g_noalloc_part));
    part = (double*)p;
    __atomic_store_n(&g_noalloc_ptr[dev], part, __ATOMIC_RELEASE);
  }
  BTA_CUDA_OK(launch_skinny_nn(P, K, J, R, ldr, M, ldm, tri, alpha, beta, in, ldin, out, ldo, part,
                               (cudaStream_t)stream));
  return BTA_OK;
}

extern "C" int bta_rows_times_block(int P, int K, int J, const double* R, int ldr, const double* M, int ldm, int tri,
                                    double alpha, double beta, const double* in, int ldin, double* out, int ldo,
                                    double* part, void* stream) {
  if (int rc = rows_times_block_check("bta_rows_times_block", P, K, J, R, M, in, beta, out); rc != BTA_OK) return rc;
  if (!part) {
    bta_set_error("bta_rows_times_block: null scratch (ceil(K/128) * P * J doubles)");
    return BTA_ERR_ARG;
  }
  BTA_CUDA_OK(launch_skinny_nn(P, K, J, R, ldr, M, ldm, tri, alpha, beta, in, ldin, out, ldo, part,
                               (cudaStream_t)stream));
  return BTA_OK;
}

extern "C" int bta_rows_times_block_t(int P, int J, int K, const double* R, int ldr, const double* M, int ldm, int tri,
                                      double alpha, double beta, const double* in, int ldin, double* out, int ldo,
                                      void* stream) {
  if (P < 1 || P > 16 || K < 1 || J < 1 || !R || !M || !out || (beta != 0.0 && !in)) {
    bta_set_error("bta_rows_times_block_t: need 1 <= P <= 16, K >= 1, J >= 1, non-null R, M, out (and in when beta != 0)");
    return BTA_ERR_ARG;
  }
  BTA_CUDA_OK(launch_skinny_nt(P, J, K, R, ldr, M, ldm, tri, alpha, beta, in, ldin, out, ldo, (cudaStream_t)stream));
  return BTA_OK;
}
