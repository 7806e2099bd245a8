// Model setup and bta_assemble (a1): Q_p(theta) from Kronecker sums of temporal and
// spatial base matrices, Q_c = Q_p + sum_v tau_v A_v^T A_v, r = sum_v tau_v A_v^T y_v (
// Eq. 10 with the coregional weights of reading R12).  Dense blocks are written straight to HBM
// (write-bound: b^2 * 8 bytes per block); the stencils are generated on the fly from grid coordinates.
#include "common.cuh"
#include "stencil.cuh"

namespace {

__global__ void theta_prep_kernel(const double* __restrict__ theta, DevParams* __restrict__ P, int k) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const int d = 3 * k + k * (k - 1) / 2 + k;
  for (int i = 0; i < d; ++i) P->theta[i] = theta[i];
  for (int m = 0; m < k; ++m)
    for (int c = 0; c < 3; ++c) P->E[m][c] = exp(theta[3 * m + c]);
  int p = 3 * k;
  for (int i = 0; i < KMAX; ++i)
    for (int j = 0; j < KMAX; ++j) P->Lam[i][j] = (i == j) ? 1.0 : 0.0;
  for (int i = 0; i < k; ++i)
    for (int j = 0; j < i; ++j) P->Lam[i][j] = theta[p++];
  for (int v = 0; v < k; ++v) P->tau[v] = exp(theta[p + v]);
  for (int c = 0; c < 3; ++c)
    for (int i = 0; i < k; ++i)
      for (int j = 0; j < k; ++j) {
        double s = 0.0;
        for (int m = 0; m < k; ++m) s += P->E[m][c] * P->Lam[m][i] * P->Lam[m][j];
        P->W[c][i][j] = s;
      }
}

// Dense blocks from stencils.  kind 0: D_t (lower triangle + diagonal, strict upper = 0; + tau cnt on the diagonal for
// Q_c);  kind 1: B_t.  Block z of a launch is global block t0 + tdir * z; tr: the transposed block (B_t^T).
// Written as a stencil band into ZEROED memory: one thread per (row i, sub-block column vj, stencil
// entry q of the 13-point pattern |dy| + |dx| <= 2) -- 13 k b entries per block instead of b^2 predicate evaluations;
// the zeros come from a memset at the full HBM write rate.
__global__ void __launch_bounds__(256) assemble_band_kernel(ModelDims md, const DevParams* __restrict__ P, int kind,
                                                            int cond, const double* __restrict__ cnt,
                                                            double* __restrict__ out, long long stride, int t0, int tdir,
                                                            int tr) {
  const long long e = (long long)blockIdx.x * 256 + threadIdx.x;
  const int per_row = 13 * md.k;
  if (e >= (long long)md.b * per_row) return;
  const int t = t0 + tdir * (int)blockIdx.y;
  const int i = (int)(e / per_row), r = (int)(e % per_row), vj = r / 13, q = r % 13;
  // q -> (dy, dx): rows dy = -2 (1 entry), -1 (3), 0 (5), 1 (3), 2 (1)
  int dy, dx;
  if (q == 0) { dy = -2; dx = 0; }
  else if (q < 4) { dy = -1; dx = q - 2; }
  else if (q < 9) { dy = 0; dx = q - 6; }
  else if (q < 12) { dy = 1; dx = q - 10; }
  else { dy = 2; dx = 0; }
  const int vi = i / md.ns, si = i % md.ns, yi = si / md.g, xi = si % md.g;
  const int yj = yi + dy, xj = xi + dx;
  if (yj < 0 || yj >= md.g || xj < 0 || xj >= md.g) return;
  const int j = vj * md.ns + yj * md.g + xj;
  // (i, j) index the block as the sweeps see it; the matrix entry is (ii, jj) (transposed coupling blocks swap them)
  if (kind == 0 && j > i) return;
  const int vii = tr ? vj : vi, vjj = tr ? vi : vj;
  const int yii = tr ? yj : yi, xii = tr ? xj : xi, yjj = tr ? yi : yj, xjj = tr ? xi : xj;
  double kv[3], mw[3];
  st_K(md.g, md.h, yii, xii, yjj, xjj, kv);
  if (kind == 0)
    st_Mdiag(md.nt, t, mw);
  else
    st_Moff(mw);
  double v = 0.0;
#pragma unroll
  for (int c = 0; c < 3; ++c) v += mw[c] * P->W[c][vii][vjj] * kv[c];
  if (kind == 0 && cond && i == j) v += P->tau[vi] * cnt[(long long)t * md.b + i];
  out[(long long)blockIdx.y * stride + (long long)i * md.b + j] = v;
}

__global__ void assemble_arrow_kernel(ModelDims md, const DevParams* __restrict__ P, int cond,
                                      const double* __restrict__ zsum, const double* __restrict__ ysum,
                                      double* __restrict__ C, long long c_stride, double* __restrict__ rhs,
                                      long long rhs_stride) {
  const int j = blockIdx.x * 256 + threadIdx.x, t = blockIdx.y;
  if (j >= md.b) return;
  const double tau = cond ? P->tau[j / md.ns] : 0.0;
  if (C)
    for (int p = 0; p < md.a; ++p)
      C[(long long)t * c_stride + (long long)p * md.b + j] =
          cond ? tau * zsum[((long long)t * md.a + p) * md.b + j] : 0.0;
  if (rhs) rhs[(long long)t * rhs_stride + j] = cond ? tau * ysum[(long long)t * md.b + j] : 0.0;
}

__global__ void assemble_tip_kernel(ModelDims md, const DevParams* __restrict__ P, int cond,
                                    const double* __restrict__ ZZ, const double* __restrict__ zy,
                                    double* __restrict__ T, int ldt, double* __restrict__ rhs_tip, int tip_stride) {
  const int p = threadIdx.x / md.a, q = threadIdx.x % md.a;
  if (p >= md.a) return;
  if (T) {
    double v = (p == q) ? md.fixed_prec : 0.0;
    if (cond)
      for (int vv = 0; vv < md.k; ++vv) v += P->tau[vv] * ZZ[(vv * md.a + p) * md.a + q];
    T[p * ldt + q] = v;
  }
  if (rhs_tip && q == 0) {
    double v = 0.0;
    if (cond)
      for (int vv = 0; vv < md.k; ++vv) v += P->tau[vv] * zy[vv * md.a + p];
    rhs_tip[p * tip_stride] = v;
  }
}

// ---------------- model setup: observation aggregates, deterministic order ----------------
__global__ void site_count_kernel(long long m, ModelDims md, const int* var, const int* node, const int* time,
                                  int* count) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= m) return;
  atomicAdd(&count[(long long)time[i] * md.b + var[i] * md.ns + node[i]], 1);
}

__global__ void __launch_bounds__(1024) site_scan_kernel(long long S, const int* count, int* start) {
  __shared__ long long sums[1024];
  const long long chunk = (S + 1023) / 1024;
  const long long lo = min(S, threadIdx.x * chunk), hi = min(S, lo + chunk);
  long long s = 0;
  for (long long e = lo; e < hi; ++e) s += count[e];
  sums[threadIdx.x] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    long long run = 0;
    for (int q = 0; q < 1024; ++q) {
      long long v = sums[q];
      sums[q] = run;
      run += v;
    }
  }
  __syncthreads();
  long long run = sums[threadIdx.x];
  for (long long e = lo; e < hi; ++e) {
    start[e] = (int)run;
    run += count[e];
  }
  if (threadIdx.x == 1023) start[S] = (int)run;
}

__global__ void site_fill_kernel(long long m, ModelDims md, const int* var, const int* node, const int* time,
                                 const int* start, int* cursor, int* idx) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= m) return;
  long long s = (long long)time[i] * md.b + var[i] * md.ns + node[i];
  int pos = atomicAdd(&cursor[s], 1);
  idx[start[s] + pos] = (int)i;
}

// In-place heapsort of idx[lo, hi) (ascending; the keys are distinct row indices, so the result is unique):
// O(n log n) for a site with n observations -- station data can put 1e5 rows on one site.
__device__ void sort_rows(int* idx, int lo, int hi) {
  const int n = hi - lo;
  int* a = idx + lo;
  auto sift = [&](int root, int end) {
    const int v = a[root];
    for (;;) {
      int ch = 2 * root + 1;
      if (ch >= end) break;
      if (ch + 1 < end && a[ch + 1] > a[ch]) ++ch;
      if (a[ch] <= v) break;
      a[root] = a[ch];
      root = ch;
    }
    a[root] = v;
  };
  for (int r = n / 2 - 1; r >= 0; --r) sift(r, n);
  for (int end = n - 1; end > 0; --end) {
    const int t = a[0];
    a[0] = a[end];
    a[end] = t;
    sift(0, end);
  }
}

// One thread per latent site: sort its observation list by row index (fixed summation order), then sum.
__global__ void site_reduce_kernel(ModelDims md, const int* start, int* idx, const int* var,
                                   const double* __restrict__ cov, const double* __restrict__ y,
                                   double* __restrict__ cnt, double* __restrict__ zsum, double* __restrict__ ysum) {
  const long long S = (long long)md.nt * md.b;
  long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= S) return;
  const int lo = start[s], hi = start[s + 1];
  if (hi - lo > 1) sort_rows(idx, lo, hi);
  const long long t = s / md.b;
  const int j = (int)(s % md.b);
  double ys = 0.0, zs[AMAX];
  for (int p = 0; p < md.apr; ++p) zs[p] = 0.0;
  for (int e = lo; e < hi; ++e) {
    const int i = idx[e];
    ys += y[i];
    for (int p = 0; p < md.apr; ++p) zs[p] += cov[(long long)i * md.apr + p];
  }
  cnt[s] = (double)(hi - lo);
  ysum[s] = ys;
  const int vv = j / md.ns;
  for (int p = 0; p < md.a; ++p) {
    const int pl = p - vv * md.apr;
    zsum[(t * md.a + p) * md.b + j] = (pl >= 0 && pl < md.apr) ? zs[pl] : 0.0;
  }
}

// grid (nvals, k): value index -> (p,q) of Z^T Z | p of Z^T y | y^T y | count, over rows of variable v
__global__ void __launch_bounds__(256) var_reduce_kernel(long long m, ModelDims md, const int* var,
                                                         const double* __restrict__ cov,
                                                         const double* __restrict__ y, double* ZZ, double* zy,
                                                         double* yy, double* mv) {
  __shared__ double red[256];
  const int val = blockIdx.x, v = blockIdx.y, apr = md.apr;
  double s = 0.0;
  for (long long i = threadIdx.x; i < m; i += 256) {
    if (var[i] != v) continue;
    double t;
    if (val < apr * apr)
      t = cov[i * apr + val / apr] * cov[i * apr + val % apr];
    else if (val < apr * apr + apr)
      t = cov[i * apr + (val - apr * apr)] * y[i];
    else if (val == apr * apr + apr)
      t = y[i] * y[i];
    else
      t = 1.0;
    s += t;
  }
  red[threadIdx.x] = s;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const double r = red[0];
    if (val < apr * apr)
      ZZ[(v * md.a + v * apr + val / apr) * md.a + v * apr + val % apr] = r;
    else if (val < apr * apr + apr)
      zy[v * md.a + v * apr + (val - apr * apr)] = r;
    else if (val == apr * apr + apr)
      yy[v] = r;
    else
      mv[v] = r;
  }
}

}  // namespace

cudaError_t launch_theta_prep(bta_ctx* c, cudaStream_t st) {
  theta_prep_kernel<<<1, 32, 0, st>>>(c->theta_dev, c->P, c->md.k);
  BTA_COUNT(c);
  return cudaGetLastError();
}

cudaError_t launch_assemble(bta_ctx* c, int which, double* D, long long d_stride, double* B, long long b_stride,
                            double* C, long long c_stride, double* T, int ldt, double* rhs, long long rhs_stride,
                            double* rhs_tip, int rhs_tip_stride, cudaStream_t st) {
  const ModelDims& md = c->md;
  const int cond = which == BTA_COND;
  if (D) {
    cudaError_t e = launch_assemble_seq(c, which, 0, 0, 1, md.nt, 0, D, d_stride, st);
    if (e != cudaSuccess) return e;
  }
  if (B && md.nt > 1) {
    cudaError_t e = launch_assemble_seq(c, which, 1, 0, 1, md.nt - 1, 0, B, b_stride, st);
    if (e != cudaSuccess) return e;
  }
  KTimeScope kt(BTA_KC_ASSEMBLE, st, 0.0, C ? 8.0 * md.a * (double)md.b * md.nt : 0.0);
  if (C || rhs) {
    dim3 ga((md.b + 255) / 256, md.nt);
    assemble_arrow_kernel<<<ga, 256, 0, st>>>(md, c->P, cond, c->zsum, c->ysum, C, c_stride, rhs, rhs_stride);
    BTA_COUNT(c);
  }
  if ((T || rhs_tip) && md.a > 0) {
    assemble_tip_kernel<<<1, md.a * md.a, 0, st>>>(md, c->P, cond, c->ZZ, c->zy, T, ldt, rhs_tip, rhs_tip_stride);
    BTA_COUNT(c);
  }
  return cudaGetLastError();
}

cudaError_t launch_assemble_block(bta_ctx* c, int which, int kind, int t, int transpose, double* out,
                                  cudaStream_t st) {
  return launch_assemble_seq(c, which, kind, t, 1, 1, transpose, out, 0, st);
}

cudaError_t launch_assemble_seq(bta_ctx* c, int which, int kind, int t0, int tdir, int count, int transpose,
                                double* out, long long stride, cudaStream_t st) {
  if (count <= 0) return cudaSuccess;
  const ModelDims& md = c->md;
  const long long bb = (long long)md.b * md.b;
  KTimeScope kt(BTA_KC_ASSEMBLE, st, 0.0, 8.0 * (double)bb * count);
  // zeros at the memset rate (contiguous blocks: one call), then the stencil band
  if (count == 1 || stride == bb || stride == -bb) {
    double* lo = (stride < 0) ? out + (long long)(count - 1) * stride : out;
    cudaError_t e = cudaMemsetAsync(lo, 0, (size_t)bb * count * sizeof(double), st);
    if (e != cudaSuccess) return e;
  } else {
    for (int z = 0; z < count; ++z) {
      cudaError_t e = cudaMemsetAsync(out + (long long)z * stride, 0, (size_t)bb * sizeof(double), st);
      if (e != cudaSuccess) return e;
    }
  }
  const long long per_block = (long long)md.b * 13 * md.k;
  dim3 g1((unsigned)((per_block + 255) / 256), count);
  assemble_band_kernel<<<g1, 256, 0, st>>>(md, c->P, kind, which == BTA_COND, c->cnt, out, stride, t0, tdir, transpose);
  BTA_COUNT(c);
  return cudaGetLastError();
}

cudaError_t run_setup_aggregates(bta_ctx* c, cudaStream_t st) {
  const ModelDims& md = c->md;
  const long long S = (long long)md.nt * md.b, m = c->m;
  int *count = nullptr, *start = nullptr, *cursor = nullptr, *idx = nullptr;
  cudaError_t e;
  auto release = [&]() {
    cudaFree(count);
    cudaFree(start);
    cudaFree(cursor);
    cudaFree(idx);
  };
  if ((e = cudaMalloc(&count, (S + 1) * sizeof(int))) != cudaSuccess || (e = cudaMalloc(&start, (S + 1) * sizeof(int))) != cudaSuccess ||
      (e = cudaMalloc(&cursor, (S + 1) * sizeof(int))) != cudaSuccess || (e = cudaMalloc(&idx, (m + 1) * sizeof(int))) != cudaSuccess) {
    release();
    return e;
  }
  cudaMemsetAsync(count, 0, (S + 1) * sizeof(int), st);
  cudaMemsetAsync(cursor, 0, (S + 1) * sizeof(int), st);
  cudaMemsetAsync(c->ZZ, 0, sizeof(double) * md.k * md.a * md.a, st);
  cudaMemsetAsync(c->zy, 0, sizeof(double) * md.k * md.a, st);
  cudaMemsetAsync(c->yy, 0, sizeof(double) * md.k, st);
  cudaMemsetAsync(c->mv, 0, sizeof(double) * md.k, st);
  if (m > 0) {
    unsigned gm = (unsigned)((m + 255) / 256);
    site_count_kernel<<<gm, 256, 0, st>>>(m, md, c->o_var, c->o_node, c->o_time, count);
    site_scan_kernel<<<1, 1024, 0, st>>>(S, count, start);
    site_fill_kernel<<<gm, 256, 0, st>>>(m, md, c->o_var, c->o_node, c->o_time, start, cursor, idx);
    c->launches += 3;
  } else {
    cudaMemsetAsync(start, 0, (S + 1) * sizeof(int), st);
  }
  site_reduce_kernel<<<(unsigned)((S + 127) / 128), 128, 0, st>>>(md, start, idx, c->o_var, c->o_cov, c->o_y, c->cnt,
                                                                 c->zsum, c->ysum);
  BTA_COUNT(c);
  if (m > 0) {
    dim3 gv(md.apr * md.apr + md.apr + 2, md.k);
    var_reduce_kernel<<<gv, 256, 0, st>>>(m, md, c->o_var, c->o_cov, c->o_y, c->ZZ, c->zy, c->yy, c->mv);
    BTA_COUNT(c);
  }
  e = cudaStreamSynchronize(st);
  release();
  if (e != cudaSuccess) return e;
  return cudaGetLastError();
}
