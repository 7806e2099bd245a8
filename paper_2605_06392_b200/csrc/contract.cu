// Gradient contractions and scalar assembly.
//   Phase A / C (Eq. 7): per-block traces <Z, dQ/dtheta> reduced to the k*k*3 partial
//     traces <Z^(ij), K_c> (Eqs. 10-12: every block Jacobian is a weight times M_c (x) K_c), gathered from the
//     <= 13 stencil entries per row of each sub-block;
//   Phase B (Eq. 9): the same bilinear forms with x*;
//   log-determinants, residual ||y - A x*||^2, and f (Eq. 1), grad f (Eq. 6).
// Every reduction has a fixed order (per-CTA tree, then a serial sum over per-CTA partials): no float atomics.
#include "common.cuh"
#include "stencil.cuh"

SmallLayout small_layout(const ModelDims& md) {
  SmallLayout L;
  L.nx = (md.ns + 255) / 256;
  size_t off = 0;
  auto take = [&](size_t n) {
    size_t o = off;
    off += (n + 31) / 32 * 32;
    return o;
  };
  const size_t tr = (size_t)md.nt * 2 * md.k * md.k * L.nx * 3;
  L.trc[0] = take(tr);
  L.trc[1] = take(tr);
  L.qd = take(tr);
  L.noise = take((size_t)md.nt * md.k * L.nx);
  L.ldpart[0] = take(64);
  L.ldpart[1] = take(64);
  L.rsspart = take(256 * md.k);
  for (int ch = 0; ch < 2; ++ch) {
    L.Tt[ch] = take(md.a * (md.a + 1));
    L.LT[ch] = take(md.a * md.a);
    L.zT[ch] = take(md.a);
    L.xT[ch] = take(md.a);
    L.ZT[ch] = take(md.a * md.a);
  }
  L.out = take(1 + md.d + 2 + 3 * md.d + md.k + 1);
  L.total = off;
  return L;
}

namespace {

// Sum over the 256 threads of a CTA in a fixed order: warp-shuffle butterflies, one shared-memory stage for the eight
// warp sums, a second butterfly in warp 0.  The result is valid in warp 0 (the callers use thread 0).
__device__ __forceinline__ double block_sum_256(double v, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  double r = 0.0;
  if (threadIdx.x < 32) {
    r = threadIdx.x < 8 ? red[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
  }
  __syncthreads();  // `red` may be reused by the next sum
  return r;
}

// grid (nx, k, k): sub-block (vi, vj) of the b x b block Z; out[((vi*k+vj)*nx + bx)*3 + c]
__global__ void __launch_bounds__(256) trace_stencil_kernel(ModelDims md, const double* __restrict__ Z, int ld,
                                                            double* __restrict__ out) {
  __shared__ double red[256];
  const int s = blockIdx.x * 256 + threadIdx.x, vi = blockIdx.y, vj = blockIdx.z, g = md.g;
  double acc[3] = {0.0, 0.0, 0.0};
  if (s < md.ns) {
    const int y = s / g, x = s % g;
    const double* zrow = Z + (long long)(vi * md.ns + s) * ld + vj * md.ns;
    for (int dy = -2; dy <= 2; ++dy)
      for (int dx = -2 + abs(dy); dx <= 2 - abs(dy); ++dx) {
        const int y2 = y + dy, x2 = x + dx;
        if (y2 < 0 || y2 >= g || x2 < 0 || x2 >= g) continue;
        double kv[3];
        st_K(g, md.h, y, x, y2, x2, kv);
        const double z = zrow[y2 * g + x2];
#pragma unroll
        for (int c = 0; c < 3; ++c) acc[c] = fma(z, kv[c], acc[c]);
      }
  }
  double* o = out + ((size_t)(vi * md.k + vj) * gridDim.x + blockIdx.x) * 3;
  for (int c = 0; c < 3; ++c) {
    double r = block_sum_256(acc[c], red);
    if (threadIdx.x == 0) o[c] = r;
  }
}

// grid (nx, k*k, nt*2): kind 0: u = x_t, v = x_t;  kind 1 (t < nt-1): u = x_{t+1}, v = x_t  (Eq. 9, R7)
__global__ void __launch_bounds__(256) quad_stencil_kernel(ModelDims md, const double* __restrict__ xv, int t_lo,
                                                           int t_hi, double* __restrict__ out) {
  __shared__ double red[256];
  const int s = blockIdx.x * 256 + threadIdx.x, vi = blockIdx.y / md.k, vj = blockIdx.y % md.k, g = md.g;
  const int t = blockIdx.z >> 1, kind = blockIdx.z & 1;
  double acc[3] = {0.0, 0.0, 0.0};
  const bool live = !(kind == 1 && t >= md.nt - 1) && t >= t_lo && t <= t_hi;
  if (live && s < md.ns) {
    const int y = s / g, x = s % g;
    const double u = xv[(long long)(t + kind) * md.b + vi * md.ns + s];
    const double* v = xv + (long long)t * md.b + vj * md.ns;
    for (int dy = -2; dy <= 2; ++dy)
      for (int dx = -2 + abs(dy); dx <= 2 - abs(dy); ++dx) {
        const int y2 = y + dy, x2 = x + dx;
        if (y2 < 0 || y2 >= g || x2 < 0 || x2 >= g) continue;
        double kv[3];
        st_K(g, md.h, y, x, y2, x2, kv);
        const double z = u * v[y2 * g + x2];
#pragma unroll
        for (int c = 0; c < 3; ++c) acc[c] = fma(z, kv[c], acc[c]);
      }
  }
  double* o = out + ((((size_t)t * 2 + kind) * md.k * md.k + blockIdx.y) * gridDim.x + blockIdx.x) * 3;
  for (int c = 0; c < 3; ++c) {
    double r = block_sum_256(acc[c], red);
    if (threadIdx.x == 0) o[c] = r;
  }
}

// grid (nx, k): sum_j in variable v of  Z_D[j][j] cnt[t][j] + 2 sum_p Z_C[p][j] zsum[t][p][j]   (Eq. 7 on tau A^T A)
__global__ void __launch_bounds__(256) noise_trace_kernel(ModelDims md, int t, const double* __restrict__ ZD, int ld,
                                                          const double* __restrict__ ZC, int ldzc,
                                                          const double* __restrict__ cnt,
                                                          const double* __restrict__ zsum, double* __restrict__ out) {
  __shared__ double red[256];
  const int s = blockIdx.x * 256 + threadIdx.x, v = blockIdx.y;
  double acc = 0.0;
  if (s < md.ns) {
    const int j = v * md.ns + s;
    acc = ZD[(long long)j * ld + j] * cnt[(long long)t * md.b + j];
    for (int p = 0; p < md.a; ++p)
      acc = fma(2.0 * ZC[(long long)p * ldzc + j], zsum[((long long)t * md.a + p) * md.b + j], acc);
  }
  double r = block_sum_256(acc, red);
  if (threadIdx.x == 0) out[((size_t)t * md.k + v) * gridDim.x + blockIdx.x] = r;
}

__global__ void __launch_bounds__(256) logdet_partial_kernel(long long N, const double* __restrict__ dvec,
                                                             double* __restrict__ out) {
  __shared__ double red[256];
  const long long chunk = (N + gridDim.x - 1) / gridDim.x;
  const long long lo = min(N, (long long)blockIdx.x * chunk), hi = min(N, lo + chunk);
  double acc = 0.0;
  for (long long e = lo + threadIdx.x; e < hi; e += 256) acc += log(dvec[e]);
  double r = block_sum_256(acc, red);
  if (threadIdx.x == 0) out[blockIdx.x] = r;
}

__global__ void __launch_bounds__(256) residual_kernel(long long m, ModelDims md, const int* __restrict__ var,
                                                       const int* __restrict__ node, const int* __restrict__ time,
                                                       const double* __restrict__ cov, const double* __restrict__ y,
                                                       const double* __restrict__ x, int t_lo, int t_hi,
                                                       double* __restrict__ out) {
  __shared__ double red[256];
  const long long chunk = (m + gridDim.x - 1) / gridDim.x;
  const long long lo = min(m, (long long)blockIdx.x * chunk), hi = min(m, lo + chunk);
  double acc[KMAX] = {0.0, 0.0, 0.0, 0.0};
  const double* xT = x + (long long)md.nt * md.b;
  for (long long i = lo + threadIdx.x; i < hi; i += 256) {
    const int v = var[i], ti = time[i];
    if (ti < t_lo || ti > t_hi) continue;
    double pred = x[(long long)ti * md.b + v * md.ns + node[i]];
    for (int p = 0; p < md.apr; ++p) pred = fma(cov[i * md.apr + p], xT[v * md.apr + p], pred);
    const double r = y[i] - pred;
#pragma unroll
    for (int q = 0; q < KMAX; ++q)
      if (q == v) acc[q] = fma(r, r, acc[q]);
  }
  for (int q = 0; q < md.k; ++q) {
    double r = block_sum_256(acc[q], red);
    if (threadIdx.x == 0) out[blockIdx.x * md.k + q] = r;
  }
}

// f (Eq. 1; readings R1, R2, R20) and grad f (Eq. 6) from the partial sums.  One CTA.
struct ScalarArgs {
  ModelDims md;
  SmallLayout L;
  const DevParams* P;
  double* small;
  const double *ZZ, *mv;
};

// theta-derivative of sum_c sum_ij W_c[i][j] T[c][i][j] for hyperparameter jj < 3k + k(k-1)/2 (Eqs. 11, 12)
__device__ double weight_contract(const ScalarArgs& A, const double* T /*[3][k][k]*/, int jj) {
  const int k = A.md.k;
  const DevParams* P = A.P;
  if (jj < 3 * k) {
    const int m = jj / 3, c = jj % 3;
    double s = 0.0;
    for (int i = 0; i < k; ++i)
      for (int j = 0; j < k; ++j) s += P->Lam[m][i] * P->Lam[m][j] * T[(c * k + i) * k + j];
    return P->E[m][c] * s;
  }
  int idx = jj - 3 * k, a = 1, b = 0;  // (a, b) enumerates (1,0), (2,0), (2,1), ...
  while (idx > 0) {
    ++b;
    if (b == a) {
      ++a;
      b = 0;
    }
    --idx;
  }
  double s = 0.0;
  for (int c = 0; c < 3; ++c)
    for (int i = 0; i < k; ++i) s += P->E[a][c] * P->Lam[a][i] * (T[(c * k + i) * k + b] + T[(c * k + b) * k + i]);
  return s;
}

__global__ void __launch_bounds__(160) scalars_kernel(ScalarArgs A) {
  __shared__ double Tsum[3][3 * KMAX * KMAX];  // [Tc | Tp | Tx][c][i][j]
  const ModelDims& md = A.md;
  const int k = md.k, nt = md.nt, nx = A.L.nx, d = md.d;
  const int e = threadIdx.x;
  if (e < 3 * 3 * k * k) {
    const int which = e / (3 * k * k), r = e % (3 * k * k), c = r / (k * k), i = (r / k) % k, j = r % k;
    const double* src = A.small + (which == 0 ? A.L.trc[CH_COND] : which == 1 ? A.L.trc[CH_PRIOR] : A.L.qd);
    double tot = 0.0;
    for (int t = 0; t < nt; ++t) {
      double mdg[3], mof[3];
      st_Mdiag(nt, t, mdg);
      st_Moff(mof);
      double sD = 0.0, sB = 0.0;
      const double* pD = src + ((((size_t)t * 2 + 0) * k + i) * k + j) * nx * 3;
      for (int bx = 0; bx < nx; ++bx) sD += pD[bx * 3 + c];
      if (t < nt - 1) {
        const double* pB1 = src + ((((size_t)t * 2 + 1) * k + i) * k + j) * nx * 3;
        const double* pB2 = src + ((((size_t)t * 2 + 1) * k + j) * k + i) * nx * 3;
        for (int bx = 0; bx < nx; ++bx) sB += pB1[bx * 3 + c] + pB2[bx * 3 + c];
      }
      tot += mdg[c] * sD + mof[c] * sB;
    }
    Tsum[which][r] = tot;
  }
  __syncthreads();
  if (threadIdx.x != 0) return;
  const DevParams* P = A.P;
  double* out = A.small + A.L.out;
  double ld[2];
  for (int ch = 0; ch < 2; ++ch) {
    double s = 0.0;
    for (int q = 0; q < 64; ++q) s += A.small[A.L.ldpart[ch] + q];
    ld[ch] = 2.0 * s;
  }
  double rss[KMAX], noiseA[KMAX];
  const double* xT = A.small + A.L.xT[CH_COND];
  const double* ZT = A.small + A.L.ZT[CH_COND];
  for (int v = 0; v < k; ++v) {
    double s = 0.0;
    for (int q = 0; q < 256; ++q) s += A.small[A.L.rsspart + q * k + v];
    rss[v] = s;
    double n = 0.0;
    for (int t = 0; t < nt; ++t)
      for (int bx = 0; bx < nx; ++bx) n += A.small[A.L.noise + ((size_t)t * k + v) * nx + bx];
    for (int p = 0; p < md.a; ++p)
      for (int q = 0; q < md.a; ++q) n += ZT[p * md.a + q] * A.ZZ[(v * md.a + p) * md.a + q];
    noiseA[v] = P->tau[v] * n;
  }
  double quad = 0.0;
  for (int c = 0; c < 3; ++c)
    for (int i = 0; i < k; ++i)
      for (int j = 0; j < k; ++j) quad += P->W[c][i][j] * Tsum[2][(c * k + i) * k + j];
  for (int p = 0; p < md.a; ++p) quad += md.fixed_prec * xT[p] * xT[p];
  const int nprior = 3 * k + k * (k - 1) / 2;
  double th2 = 0.0;
  for (int j = 0; j < d; ++j) th2 += P->theta[j] * P->theta[j];
  double f = -0.5 * th2 + 0.5 * ld[CH_PRIOR] - 0.5 * ld[CH_COND] - 0.5 * quad;
  for (int v = 0; v < k; ++v) f += 0.5 * A.mv[v] * P->theta[nprior + v] - 0.5 * P->tau[v] * rss[v];
  double* grad = out + 1;
  double* ldo = out + 1 + d;
  double* parts = out + 1 + d + 2;
  double* rsso = parts + 3 * d;
  for (int j = 0; j < nprior; ++j) {
    const double a_ = weight_contract(A, Tsum[0], j), c_ = weight_contract(A, Tsum[1], j),
                 b_ = weight_contract(A, Tsum[2], j);
    parts[j] = a_;
    parts[d + j] = b_;
    parts[2 * d + j] = c_;
    grad[j] = -0.5 * a_ - 0.5 * b_ + 0.5 * c_ - P->theta[j];
  }
  for (int v = 0; v < k; ++v) {
    const int j = nprior + v;
    parts[j] = noiseA[v];
    parts[d + j] = 0.0;
    parts[2 * d + j] = 0.0;
    grad[j] = -0.5 * noiseA[v] + 0.5 * A.mv[v] - 0.5 * P->tau[v] * rss[v] - P->theta[j];
    rsso[v] = rss[v];
  }
  out[0] = f;
  ldo[0] = ld[CH_PRIOR];
  ldo[1] = ld[CH_COND];
  rsso[k] = quad;
}

}  // namespace

cudaError_t launch_trace_stencil(bta_ctx* c, int chain, int t, int kind, const double* Z, int ld, cudaStream_t st) {
  const ModelDims& md = c->md;
  SmallLayout L = small_layout(md);
  double* out = c->small + L.trc[chain] + ((size_t)t * 2 + kind) * md.k * md.k * L.nx * 3;
  dim3 grid(L.nx, md.k, md.k);
  // bytes: the <= 13 gathered entries of every row of every sub-block (payload, not sectors)
  KTimeScope kt(BTA_KC_CONTRACT, st, 6.0 * 13.0 * md.k * (double)md.b, 8.0 * 13.0 * md.k * (double)md.b);
  trace_stencil_kernel<<<grid, 256, 0, st>>>(md, Z, ld, out);
  BTA_COUNT(c);
  return cudaGetLastError();
}

cudaError_t launch_noise_trace(bta_ctx* c, int t, const double* ZD, int ld, const double* ZC, int ldzc,
                               cudaStream_t st) {
  const ModelDims& md = c->md;
  SmallLayout L = small_layout(md);
  dim3 grid(L.nx, md.k);
  KTimeScope kt(BTA_KC_CONTRACT, st, 2.0 * (1 + md.a) * (double)md.b, 8.0 * 2.0 * (1 + md.a) * (double)md.b);
  noise_trace_kernel<<<grid, 256, 0, st>>>(md, t, ZD, ld, ZC, ldzc, c->cnt, c->zsum, c->small + L.noise);
  BTA_COUNT(c);
  return cudaGetLastError();
}

cudaError_t launch_quad_stencil(bta_ctx* c, const double* x, cudaStream_t st) {
  return launch_quad_stencil(c, x, 0, c->md.nt - 1, st);
}
cudaError_t launch_quad_stencil(bta_ctx* c, const double* x, int t_lo, int t_hi, cudaStream_t st) {
  const ModelDims& md = c->md;
  SmallLayout L = small_layout(md);
  dim3 grid(L.nx, md.k * md.k, md.nt * 2);
  KTimeScope kt(BTA_KC_CONTRACT, st, 2.0 * 7.0 * 13.0 * md.k * (double)md.b * md.nt, 8.0 * 2.0 * md.k * (double)md.N);
  quad_stencil_kernel<<<grid, 256, 0, st>>>(md, x, t_lo, t_hi, c->small + L.qd);
  BTA_COUNT(c);
  return cudaGetLastError();
}

cudaError_t launch_logdet_partial(bta_ctx* c, int chain, const double* dvec, cudaStream_t st) {
  SmallLayout L = small_layout(c->md);
  KTimeScope kt(BTA_KC_OTHER, st, 0.0, 8.0 * (double)c->md.N);
  logdet_partial_kernel<<<64, 256, 0, st>>>(c->md.N, dvec, c->small + L.ldpart[chain]);
  BTA_COUNT(c);
  return cudaGetLastError();
}

cudaError_t launch_residual(bta_ctx* c, const double* x, cudaStream_t st) {
  return launch_residual(c, x, 0, c->md.nt - 1, st);
}
cudaError_t launch_residual(bta_ctx* c, const double* x, int t_lo, int t_hi, cudaStream_t st) {
  SmallLayout L = small_layout(c->md);
  KTimeScope kt(BTA_KC_OTHER, st, 0.0, (double)c->m * (12.0 + 8.0 * c->md.apr + 8.0));
  residual_kernel<<<256, 256, 0, st>>>(c->m, c->md, c->o_var, c->o_node, c->o_time, c->o_cov, c->o_y, x, t_lo, t_hi,
                                       c->small + L.rsspart);
  BTA_COUNT(c);
  return cudaGetLastError();
}

cudaError_t launch_scalars(bta_ctx* c, cudaStream_t st) {
  ScalarArgs A{c->md, small_layout(c->md), c->P, c->small, c->ZZ, c->mv};
  KTimeScope kt(BTA_KC_OTHER, st, 0.0, 0.0);
  scalars_kernel<<<1, 160, 0, st>>>(A);
  BTA_COUNT(c);
  return cudaGetLastError();
}

namespace {
__global__ void logdet_final_kernel(const double* __restrict__ part, double* __restrict__ out) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double s = 0.0;
  for (int q = 0; q < 64; ++q) s += part[q];
  out[0] = 2.0 * s;
}
}  // namespace

// out[0] (device) = 2 * sum log diag(L) from the 64 partial sums of launch_logdet_partial
cudaError_t launch_logdet_final(bta_ctx* c, int chain, double* out, cudaStream_t st) {
  SmallLayout L = small_layout(c->md);
  logdet_final_kernel<<<1, 32, 0, st>>>(c->small + L.ldpart[chain], out);
  BTA_COUNT(c);
  return cudaGetLastError();
}
