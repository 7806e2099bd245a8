// The arrow tip (Algorithm 1 line 11, Eq. 3, Z_T of the selected inversion) and small helpers.  The POTRF/TRTRI leaf
// of the diagonal blocks is leaf.cu.

#include "common.cuh"

namespace {

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

cudaError_t launch_tip(const double* Tt, int a, int nr, int do_chol, double* LT, double* zT, double* xT, double* ZT,
                       double* diagL, long long grow0, unsigned long long* pivot_flag, cudaStream_t st) {
  KTimeScope kt(BTA_KC_OTHER, st, 0.0, 0.0);
  tip_kernel<<<1, 32, 0, st>>>(Tt, a, nr, do_chol, LT, zT, xT, ZT, diagL, grow0, pivot_flag);
  return cudaGetLastError();
}

cudaError_t launch_zero_upper(double* A, int ld, int n, cudaStream_t st) {
  dim3 grid((n + 255) / 256, n);
  KTimeScope kt(BTA_KC_OTHER, st, 0.0, 4.0 * n * (double)n);
  zero_upper_kernel<<<grid, 256, 0, st>>>(A, ld, n);
  return cudaGetLastError();
}

cudaError_t launch_tip_inverse(const double* LT, int a, double* ZT, cudaStream_t st) {
  tip_inverse_kernel<<<1, 32, 0, st>>>(LT, a, ZT);
  return cudaGetLastError();
}
