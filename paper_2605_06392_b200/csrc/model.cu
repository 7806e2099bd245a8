// bta_create / bta_destroy: model context, device copies of the observations, theta-independent aggregates.
#include <cstdlib>
#include <cstring>

#include <cuda.h>

#include "common.cuh"

namespace {
template <typename T>
cudaError_t dev_alloc(T** p, size_t n) {
  return cudaMalloc((void**)p, (n ? n : 1) * sizeof(T));
}
}  // namespace

// Green-context SM partition for the forward sweeps (common.cuh: s_fwd).  The driver entry points are looked up at run
// time (cudaGetDriverEntryPoint), so the library keeps no link-time dependency on libcuda.  An optimisation only: on any
// failure the partition is left off (fwd_sms = 0) and the reason goes to bta_last_error.
namespace {
template <class F>
bool drv(const char* name, F& fn) {
  void* p = nullptr;
  cudaDriverEntryPointQueryResult qr;
  if (cudaGetDriverEntryPoint(name, &p, cudaEnableDefault, &qr) != cudaSuccess || qr != cudaDriverEntryPointSuccess || !p)
    return false;
  fn = reinterpret_cast<F>(p);
  return true;
}
void make_forward_partition(bta_ctx* c, int device, int reserve, int prio) {
  CUresult (*getRes)(CUdevice, CUdevResource*, CUdevResourceType) = nullptr;
  CUresult (*split)(CUdevResource*, unsigned int*, const CUdevResource*, CUdevResource*, unsigned int, unsigned int) =
      nullptr;
  CUresult (*genDesc)(CUdevResourceDesc*, CUdevResource*, unsigned int) = nullptr;
  CUresult (*gcreate)(CUgreenCtx*, CUdevResourceDesc, CUdevice, unsigned int) = nullptr;
  CUresult (*gstream)(CUstream*, CUgreenCtx, unsigned int, int) = nullptr;
  CUresult (*devGet)(CUdevice*, int) = nullptr;
  if (!drv("cuDeviceGetDevResource", getRes) || !drv("cuDevSmResourceSplitByCount", split) ||
      !drv("cuDevResourceGenerateDesc", genDesc) || !drv("cuGreenCtxCreate", gcreate) ||
      !drv("cuGreenCtxStreamCreate", gstream) || !drv("cuDeviceGet", devGet)) {
    bta_set_error("BTA_FWD_RESERVE: green-context driver entry points not available");
    return;
  }
  CUdevice dev;
  CUdevResource all, part, rest;
  if (devGet(&dev, device) != CUDA_SUCCESS || getRes(dev, &all, CU_DEV_RESOURCE_TYPE_SM) != CUDA_SUCCESS) {
    bta_set_error("BTA_FWD_RESERVE: cuDeviceGetDevResource failed");
    return;
  }
  const int total = (int)all.sm.smCount;
  if (reserve >= total) return;
  unsigned int ngroups = 1;
  if (split(&part, &ngroups, &all, &rest, 0, (unsigned)(total - reserve)) != CUDA_SUCCESS || ngroups != 1) {
    bta_set_error("BTA_FWD_RESERVE: cuDevSmResourceSplitByCount failed");
    return;
  }
  CUdevResourceDesc desc;
  CUgreenCtx g;
  if (genDesc(&desc, &part, 1) != CUDA_SUCCESS || gcreate(&g, desc, dev, CU_GREEN_CTX_DEFAULT_STREAM) != CUDA_SUCCESS) {
    bta_set_error("BTA_FWD_RESERVE: cuGreenCtxCreate failed");
    return;
  }
  c->green_ctx = g;
  for (auto& q : c->s_fwd) {
    CUstream st = nullptr;
    if (gstream(&st, g, CU_STREAM_NON_BLOCKING, prio) != CUDA_SUCCESS) {
      bta_set_error("BTA_FWD_RESERVE: cuGreenCtxStreamCreate failed");
      for (auto& r : c->s_fwd) {
        if (r) cudaStreamDestroy(r);
        r = nullptr;
      }
      return;
    }
    q = st;
  }
  c->fwd_sms = (int)part.sm.smCount;
}
void destroy_forward_partition(bta_ctx* c) {
  if (!c->green_ctx) return;
  CUresult (*gdestroy)(CUgreenCtx) = nullptr;
  if (drv("cuGreenCtxDestroy", gdestroy)) gdestroy((CUgreenCtx)c->green_ctx);
  c->green_ctx = nullptr;
}
}  // namespace

extern "C" int bta_create(bta_ctx** out, const bta_model_desc* desc, const bta_obs* obs, int device) {
  if (!out) return BTA_ERR_ARG;
  *out = nullptr;
  if (!desc || !obs) {
    bta_set_error("bta_create: null descriptor or observations");
    return BTA_ERR_ARG;
  }
  if (desc->nt < 1 || desc->g < 1 || desc->k < 1 || desc->k > KMAX || desc->a < desc->k || desc->a > AMAX ||
      desc->a % desc->k != 0 || !(desc->h > 0.0) || !(desc->fixed_prec > 0.0) || obs->m < 0 ||
      obs->m > 2000000000LL) {
    bta_set_error("bta_create: need nt>=1, g>=1, 1<=k<=4, k<=a<=8, a%k==0, h>0, fixed_prec>0, 0<=m<2e9");
    return BTA_ERR_ARG;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
    bta_set_error("bta_create: no such CUDA device (this library has no CPU fallback)");
    return BTA_ERR_NODEVICE;
  }
  cudaDeviceProp prop;
  BTA_CUDA_OK(cudaGetDeviceProperties(&prop, device));
  if (prop.major != 10) {
    bta_set_error("bta_create: device is not sm_100-class (kernels are built for sm_100a only; no fallback)");
    return BTA_ERR_NODEVICE;
  }
  BTA_CUDA_OK(cudaSetDevice(device));
  bta_ctx* c = new bta_ctx();
  ModelDims& md = c->md;
  md.nt = desc->nt;
  md.g = desc->g;
  md.ns = desc->g * desc->g;
  md.k = desc->k;
  md.a = desc->a;
  md.apr = desc->a / desc->k;
  md.b = md.k * md.ns;
  md.d = 3 * md.k + md.k * (md.k - 1) / 2 + md.k;
  md.N = (long long)md.nt * md.b + md.a;
  md.h = desc->h;
  md.fixed_prec = desc->fixed_prec;
  c->device = device;
  c->m = obs->m;
  c->launches = 0;
  c->last_pivot = 0;
  c->last_x_dev = nullptr;
  const long long m = obs->m;
  for (long long i = 0; i < m; ++i) {
    if (obs->var[i] < 0 || obs->var[i] >= md.k || obs->node[i] < 0 || obs->node[i] >= md.ns || obs->time[i] < 0 ||
        obs->time[i] >= md.nt) {
      delete c;
      bta_set_error("bta_create: observation index out of range");
      return BTA_ERR_ARG;
    }
  }
  const size_t S = (size_t)md.nt * md.b;
  BTA_CUDA_OK(dev_alloc(&c->o_var, m));
  BTA_CUDA_OK(dev_alloc(&c->o_node, m));
  BTA_CUDA_OK(dev_alloc(&c->o_time, m));
  BTA_CUDA_OK(dev_alloc(&c->o_cov, m * md.apr));
  BTA_CUDA_OK(dev_alloc(&c->o_y, m));
  BTA_CUDA_OK(dev_alloc(&c->cnt, S));
  BTA_CUDA_OK(dev_alloc(&c->zsum, S * md.a));
  BTA_CUDA_OK(dev_alloc(&c->ysum, S));
  BTA_CUDA_OK(dev_alloc(&c->ZZ, (size_t)md.k * md.a * md.a));
  BTA_CUDA_OK(dev_alloc(&c->zy, (size_t)md.k * md.a));
  BTA_CUDA_OK(dev_alloc(&c->yy, md.k));
  BTA_CUDA_OK(dev_alloc(&c->mv, md.k));
  BTA_CUDA_OK(dev_alloc(&c->P, 1));
  BTA_CUDA_OK(dev_alloc(&c->theta_dev, DMAX));
  BTA_CUDA_OK(dev_alloc(&c->pivot_flag, 1));
  SmallLayout L = small_layout(md);
  c->small_doubles = L.total;
  BTA_CUDA_OK(dev_alloc(&c->small, L.total));
  BTA_CUDA_OK(cudaMemset(c->small, 0, L.total * sizeof(double)));
  BTA_CUDA_OK(cudaMallocHost((void**)&c->host_pinned, 4096 * sizeof(double)));
  // Optional stream priorities (BTA_PRIORITY=1): Q_c chains highest, Q_p chains lowest.  Measured: the Q_c chains
  // finish 25 % earlier but the Q_p chains are starved by the same amount -- with four chains in flight the GPU is
  // throughput-bound, so the default is equal priorities.
  int prio_lo = 0, prio_hi = 0;
  BTA_CUDA_OK(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
  {
    const char* e = getenv("BTA_PRIORITY");
    if (!(e && e[0] == '1')) prio_hi = prio_lo;
  }
  BTA_CUDA_OK(cudaStreamCreateWithPriority(&c->s_main, cudaStreamNonBlocking, prio_hi));
  BTA_CUDA_OK(cudaStreamCreateWithPriority(&c->s_aux[0], cudaStreamNonBlocking, prio_hi));
  BTA_CUDA_OK(cudaStreamCreateWithPriority(&c->s_side, cudaStreamNonBlocking, prio_lo));
  BTA_CUDA_OK(cudaStreamCreateWithPriority(&c->s_aux[1], cudaStreamNonBlocking, prio_lo));
  for (int q = 0; q < 2; ++q) {
    c->graph_exec[q] = nullptr;
    c->graph_ws[q] = nullptr;
    c->graph_launches[q] = 0;
  }
  c->grad_calls = 0;
  c->trace_on = getenv("BTA_TRACE") != nullptr;
  c->store_mode = BTA_STORE_FACTOR;
  for (auto& e : c->ev) BTA_CUDA_OK(cudaEventCreate(&e));
  {
    int plo = 0, phi = 0;
    BTA_CUDA_OK(cudaDeviceGetStreamPriorityRange(&plo, &phi));
    for (auto& q : c->s_hi) BTA_CUDA_OK(cudaStreamCreateWithPriority(&q, cudaStreamNonBlocking, phi));
    for (auto& q : c->s_x) BTA_CUDA_OK(cudaStreamCreateWithPriority(&q, cudaStreamNonBlocking, plo));
    for (auto& q : c->s_fwd) q = nullptr;
    c->green_ctx = nullptr;
    c->fwd_sms = 0;
    if (const char* e = getenv("BTA_FWD_RESERVE")) {
      const int reserve = atoi(e);
      if (reserve > 0) make_forward_partition(c, device, reserve, plo);
    }
    for (auto& e : c->ev_sw) BTA_CUDA_OK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    c->ev_sw_next = 0;
  }
  if (m > 0) {
    BTA_CUDA_OK(cudaMemcpy(c->o_var, obs->var, m * sizeof(int), cudaMemcpyHostToDevice));
    BTA_CUDA_OK(cudaMemcpy(c->o_node, obs->node, m * sizeof(int), cudaMemcpyHostToDevice));
    BTA_CUDA_OK(cudaMemcpy(c->o_time, obs->time, m * sizeof(int), cudaMemcpyHostToDevice));
    BTA_CUDA_OK(cudaMemcpy(c->o_cov, obs->cov, m * md.apr * sizeof(double), cudaMemcpyHostToDevice));
    BTA_CUDA_OK(cudaMemcpy(c->o_y, obs->y, m * sizeof(double), cudaMemcpyHostToDevice));
  }
  BTA_CUDA_OK(run_setup_aggregates(c, 0));
  *out = c;
  return BTA_OK;
}

extern "C" int bta_destroy(bta_ctx* c) {
  if (!c) return BTA_OK;
  cudaSetDevice(c->device);
  cudaFree(c->o_var);
  cudaFree(c->o_node);
  cudaFree(c->o_time);
  cudaFree(c->o_cov);
  cudaFree(c->o_y);
  cudaFree(c->cnt);
  cudaFree(c->zsum);
  cudaFree(c->ysum);
  cudaFree(c->ZZ);
  cudaFree(c->zy);
  cudaFree(c->yy);
  cudaFree(c->mv);
  cudaFree(c->P);
  cudaFree(c->theta_dev);
  cudaFree(c->pivot_flag);
  cudaFree(c->small);
  cudaFreeHost(c->host_pinned);
  for (int q = 0; q < 2; ++q)
    if (c->graph_exec[q]) cudaGraphExecDestroy(c->graph_exec[q]);
  cudaStreamDestroy(c->s_side);
  cudaStreamDestroy(c->s_main);
  for (auto& q : c->s_aux) cudaStreamDestroy(q);
  for (auto& e : c->ev) cudaEventDestroy(e);
  for (auto& q : c->s_hi) cudaStreamDestroy(q);
  for (auto& q : c->s_x) cudaStreamDestroy(q);
  for (auto& q : c->s_fwd)
    if (q) cudaStreamDestroy(q);
  destroy_forward_partition(c);
  for (auto& e : c->ev_sw) cudaEventDestroy(e);
  delete c;
  return BTA_OK;
}

extern "C" int32_t bta_num_hyper(const bta_ctx* c) { return c ? c->md.d : 0; }
extern "C" int64_t bta_latent_size(const bta_ctx* c) { return c ? c->md.N : 0; }
extern "C" int64_t bta_last_pivot(const bta_ctx* c) { return c ? c->last_pivot : 0; }
extern "C" int64_t bta_kernel_launches(const bta_ctx* c) { return c ? c->launches : 0; }

extern "C" int bta_set_store_mode(bta_ctx* c, int mode) {
  if (!c || (mode != BTA_STORE_FACTOR && mode != BTA_STORE_CARRY)) {
    bta_set_error("bta_set_store_mode: null ctx or unknown mode");
    return BTA_ERR_ARG;
  }
  for (int q = 0; q < 2; ++q)
    if (mode != c->store_mode && c->graph_exec[q]) {  // a cached graph was captured for the other layout
      cudaGraphExecDestroy(c->graph_exec[q]);
      c->graph_exec[q] = nullptr;
    }
  c->store_mode = mode;
  return BTA_OK;
}
extern "C" int bta_get_store_mode(const bta_ctx* c) { return c ? c->store_mode : -1; }
