// Leaf kernels of the blocked POTRF/TRTRI recursion and the arrow tip.
//
// potrf_inv_tile: one CTA factors an n x n (n <= 64) diagonal tile A = L L^T and inverts L in the same
// sweep, in place in shared memory: at step k the columns j <= k of the working array hold the rows of
// L^-1 built so far (forward elimination applied to the identity) and the columns j > k hold the Schur
// complement.  Output: X = L^-1 (lower; strict upper of the tile zeroed), diag(L) for the log-determinant
// (PAPER.md:48), and the first non-positive pivot (Algorithm 1 line 3 needs D_i - S_{i-1} > 0).
#include <cstdlib>

#include "common.cuh"

namespace {

// NB x NB leaf, NW warps.  Warp w owns rows w, w+NW, ... (register slot r = row / NW); lane l owns columns l,
// l+32, ... (slot c = col / 32): the whole working array lives in registers.  Elimination step k: the owners of
// column k, row k and the pivot publish them (double-buffered shared vectors) together with 1/sqrt(pivot); one
// __syncthreads; then every thread updates its registers with bare DFMAs.  The steps are generated in blocks of
// NW consecutive k (template parameter BLK) so that the register slots of column k and row k are compile-time
// constants and the per-step instruction count stays small.
template <int NB, int NW>
struct LeafSmem {
  double colraw[2][NB], rowraw[2][NB], diagraw[2];
};

struct LeafPivot {
  double rs, piv;  // 1/sqrt(pivot_k) and pivot_k, held redundantly by every thread
};

template <int NB, int NW, int BLK>
__device__ __forceinline__ bool leaf_steps(double (&w)[NB / NW][NB / 32], LeafSmem<NB, NW>& sm, LeafPivot& pv, int n,
                                           int lane, int warp, double* __restrict__ diagL, long long grow0,
                                           unsigned long long* __restrict__ pivot_flag) {
  constexpr int R = NB / NW, CC = NB / 32;
  constexpr int K0 = BLK * NW, KC = K0 / 32, KR = BLK, L0 = K0 % 32;
  constexpr int KCN = (K0 + NW) / 32;  // column slot of the first pivot of the next block
#pragma unroll 1
  for (int q = 0; q < NW; ++q) {
    const int k = K0 + q, kl = L0 + q, buf = q & 1;
    if (k >= n) return false;
    // ---- publish column k (rows >= K0), row k (columns <= k) and the raw diagonal entry of step k+1
    if (lane == kl) {
#pragma unroll
      for (int r = KR; r < R; ++r) sm.colraw[buf][warp + NW * r] = w[r][KC];
    }
    if (warp == q) {
#pragma unroll
      for (int c = 0; c <= KC; ++c) sm.rowraw[buf][lane + 32 * c] = w[KR][c];
    }
    if (q < NW - 1) {
      if (warp == q + 1 && lane == kl + 1) sm.diagraw[buf] = w[KR][KC];
    } else if (KR + 1 < R) {
      if (warp == 0 && lane == (L0 + NW) % 32) sm.diagraw[buf] = w[KR + 1 < R ? KR + 1 : KR][KCN < CC ? KCN : KC];
    }
    __syncthreads();
    const double* cr = sm.colraw[buf];
    const double* rr = sm.rowraw[buf];
    const double rs = pv.rs;
    if (threadIdx.x == 0 && diagL) diagL[k] = pv.piv * rs;
    // ---- 1/sqrt of the next pivot, by every thread, off the critical path of the updates below
    if (k + 1 < n) {
      const double l = cr[k + 1] * rs;
      double pn = fma(-l, l, sm.diagraw[buf]);
      if (!(pn > 0.0)) {  // also catches NaN
        if (threadIdx.x == 0) atomicMin(pivot_flag, (unsigned long long)(grow0 + k + 2));
        pn = 1.0;
      }
      pv.piv = pn;
      pv.rs = rsqrt(pn);
    }
    double cv[CC];
#pragma unroll
    for (int c = 0; c < CC; ++c) {
      const int j = lane + 32 * c;
      if (c < KC)
        cv[c] = rr[j] * rs;
      else if (c > KC)
        cv[c] = cr[j] * rs;
      else
        cv[c] = (lane < kl ? rr[j] : cr[j]) * rs;
    }
    if (lane == kl) {  // column k restarts: X[i][k] = -l_ik / l_kk for i > k, X[k][k] = 1 / l_kk
      cv[KC] = rs;
#pragma unroll
      for (int r = KR; r < R; ++r) w[r][KC] = 0.0;
    }
#pragma unroll
    for (int r = KR; r < R; ++r) {
      const int i = warp + NW * r;
      // columns beyond the diagonal slot of this row are never read: skip them
      const int cmax = (NW * r + NW - 1) / 32;
      if (r > KR || warp > q) {
        const double nli = -cr[i] * rs;
#pragma unroll
        for (int c = 0; c < CC; ++c)
          if (c <= cmax) w[r][c] = fma(nli, cv[c], w[r][c]);
      } else if (warp == q) {
#pragma unroll
        for (int c = 0; c <= KC; ++c)
          if (lane + 32 * c <= k) w[r][c] = cv[c];
      }
    }
  }
  return true;
}

template <int NB, int NW, int BLK>
struct LeafRun {
  static __device__ __forceinline__ void run(double (&w)[NB / NW][NB / 32], LeafSmem<NB, NW>& sm, LeafPivot& pv,
                                             int n, int lane, int warp, double* diagL, long long grow0,
                                             unsigned long long* pivot_flag) {
    if (leaf_steps<NB, NW, BLK>(w, sm, pv, n, lane, warp, diagL, grow0, pivot_flag))
      LeafRun<NB, NW, BLK + 1>::run(w, sm, pv, n, lane, warp, diagL, grow0, pivot_flag);
  }
};
template <int NB, int NW>
struct LeafRun<NB, NW, NB / NW> {
  static __device__ __forceinline__ void run(double (&)[NB / NW][NB / 32], LeafSmem<NB, NW>&, LeafPivot&, int, int,
                                             int, double*, long long, unsigned long long*) {}
};

template <int NB, int NW>
__global__ void __launch_bounds__(32 * NW) potrf_inv_tile_kernel(double* __restrict__ A, int ld, int n,
                                                                 double* __restrict__ diagL, long long grow0,
                                                                 unsigned long long* __restrict__ pivot_flag) {
  constexpr int R = NB / NW, CC = NB / 32;
  static_assert(NW % 2 == 0 && 32 % NW == 0, "steps alternate the two shared buffers inside a block of NW");
  __shared__ LeafSmem<NB, NW> sm;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  double w[R][CC];
#pragma unroll
  for (int r = 0; r < R; ++r)
#pragma unroll
    for (int c = 0; c < CC; ++c) {
      const int i = warp + NW * r, j = lane + 32 * c;
      double v = (i == j) ? 1.0 : 0.0;
      if (i < n && j <= i) v = A[(long long)i * ld + j];
      w[r][c] = v;
    }
  LeafPivot pv;
  pv.piv = A[0];
  if (!(pv.piv > 0.0)) {
    if (tid == 0) atomicMin(pivot_flag, (unsigned long long)(grow0 + 1));
    pv.piv = 1.0;
  }
  pv.rs = rsqrt(pv.piv);
  LeafRun<NB, NW, 0>::run(w, sm, pv, n, lane, warp, diagL, grow0, pivot_flag);
#pragma unroll
  for (int r = 0; r < R; ++r)
#pragma unroll
    for (int c = 0; c < CC; ++c) {
      const int i = warp + NW * r, j = lane + 32 * c;
      if (i < n && j < n) A[(long long)i * ld + j] = (j <= i) ? w[r][c] : 0.0;
    }
}

// Arrow tip (Algorithm 1 line 11, Eq. 3, and Z_T = L_T^-T L_T^-1 of the selected inversion, R10).
// Tt is [a][a+nr]: the reduced tip T~_n (lower triangle read; used when do_chol) and, in columns a..a+nr-1,
// the reduced right-hand sides r_T - v_T.  do_chol = 0: L_T is given (solve with an existing factor).
// Outputs zT[r][a], xT[r][a] per right-hand side r.  One thread: a <= 16, O(a^3) work, once per sweep.
__global__ void tip_kernel(const double* __restrict__ Tt, int a, int nr, int do_chol, double* __restrict__ LT,
                           double* __restrict__ zT, double* __restrict__ xT, double* __restrict__ ZT,
                           double* __restrict__ diagL, long long grow0, unsigned long long* pivot_flag) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const int ldt = a + nr;
  double L[16][16], Xi[16][16];
  for (int i = 0; i < a; ++i)
    for (int j = 0; j < a; ++j) {
      L[i][j] = (j <= i) ? (do_chol ? Tt[i * ldt + j] : LT[i * a + j]) : 0.0;
      Xi[i][j] = 0.0;
    }
  if (do_chol) {
    for (int k = 0; k < a; ++k) {
      double piv = L[k][k];
      for (int q = 0; q < k; ++q) piv -= L[k][q] * L[k][q];
      if (!(piv > 0.0)) {
        atomicMin(pivot_flag, (unsigned long long)(grow0 + k + 1));
        piv = 1.0;
      }
      double d = sqrt(piv);
      L[k][k] = d;
      if (diagL) diagL[k] = d;
      for (int i = k + 1; i < a; ++i) {
        double s = L[i][k];
        for (int q = 0; q < k; ++q) s -= L[i][q] * L[k][q];
        L[i][k] = s / d;
      }
    }
  }
  for (int j = 0; j < a; ++j) {  // Xi = L^-1 column by column
    Xi[j][j] = 1.0 / L[j][j];
    for (int i = j + 1; i < a; ++i) {
      double s = 0.0;
      for (int q = j; q < i; ++q) s += L[i][q] * Xi[q][j];
      Xi[i][j] = -s / L[i][i];
    }
  }
  if (do_chol) {
    for (int i = 0; i < a; ++i)
      for (int j = 0; j < a; ++j) {
        LT[i * a + j] = L[i][j];
        double s = 0.0;
        for (int q = (i > j ? i : j); q < a; ++q) s += Xi[q][i] * Xi[q][j];
        if (ZT) ZT[i * a + j] = s;
      }
  }
  for (int r = 0; r < nr; ++r) {
    double z[16];
    for (int i = 0; i < a; ++i) {
      double s = 0.0;
      for (int q = 0; q <= i; ++q) s += Xi[i][q] * Tt[q * ldt + a + r];
      z[i] = s;
      if (zT) zT[r * a + i] = s;
    }
    for (int i = 0; i < a; ++i) {
      double s = 0.0;
      for (int q = i; q < a; ++q) s += Xi[q][i] * z[q];
      xT[r * a + i] = s;
    }
  }
}

// Zero the strict upper triangle of an n x n block (the library keeps lower triangles authoritative).
__global__ void zero_upper_kernel(double* __restrict__ A, int ld, int n) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
  if (j < n && j > i) A[(long long)i * ld + j] = 0.0;
}

// Z_T from a given L_T (selected inversion started from a stored factor).
__global__ void tip_inverse_kernel(const double* __restrict__ LT, int a, double* __restrict__ ZT) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double Xi[16][16];
  for (int i = 0; i < a; ++i)
    for (int j = 0; j < a; ++j) Xi[i][j] = 0.0;
  for (int j = 0; j < a; ++j) {
    Xi[j][j] = 1.0 / LT[j * a + j];
    for (int i = j + 1; i < a; ++i) {
      double s = 0.0;
      for (int q = j; q < i; ++q) s += LT[i * a + q] * Xi[q][j];
      Xi[i][j] = -s / LT[i * a + i];
    }
  }
  for (int i = 0; i < a; ++i)
    for (int j = 0; j < a; ++j) {
      double s = 0.0;
      for (int q = (i > j ? i : j); q < a; ++q) s += Xi[q][i] * Xi[q][j];
      ZT[i * a + j] = s;
    }
}

}  // namespace

cudaError_t launch_potrf_inv_tile(double* A, int ld, int n, double* diagL, long long grow0,
                                  unsigned long long* pivot_flag, cudaStream_t st) {
  static const int blocked = [] {
    const char* e = getenv("BTA_LEAF_BLOCKED");
    return e ? atoi(e) : 1;
  }();
  if (blocked) return launch_potrf_inv_blocked(A, ld, n, diagL, grow0, pivot_flag, st);
  if (n <= 64)
    potrf_inv_tile_kernel<64, 8><<<1, 256, 0, st>>>(A, ld, n, diagL, grow0, pivot_flag);
  else if (n <= 128)
    potrf_inv_tile_kernel<128, 8><<<1, 256, 0, st>>>(A, ld, n, diagL, grow0, pivot_flag);
  else
    return cudaErrorInvalidValue;
  return cudaGetLastError();
}

cudaError_t launch_tip(const double* Tt, int a, int nr, int do_chol, double* LT, double* zT, double* xT, double* ZT,
                       double* diagL, long long grow0, unsigned long long* pivot_flag, cudaStream_t st) {
  tip_kernel<<<1, 32, 0, st>>>(Tt, a, nr, do_chol, LT, zT, xT, ZT, diagL, grow0, pivot_flag);
  return cudaGetLastError();
}

cudaError_t launch_zero_upper(double* A, int ld, int n, cudaStream_t st) {
  dim3 grid((n + 255) / 256, n);
  zero_upper_kernel<<<grid, 256, 0, st>>>(A, ld, n);
  return cudaGetLastError();
}

cudaError_t launch_tip_inverse(const double* LT, int a, double* ZT, cudaStream_t st) {
  tip_inverse_kernel<<<1, 32, 0, st>>>(LT, a, ZT);
  return cudaGetLastError();
}
