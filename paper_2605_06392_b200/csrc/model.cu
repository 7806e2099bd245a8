// bta_create / bta_destroy: model context, device copies of the observations, theta-independent aggregates.
#include <cstdlib>
#include <cstring>

#include "common.cuh"

namespace {
template <typename T>
cudaError_t dev_alloc(T** p, size_t n) {
  return cudaMalloc((void**)p, (n ? n : 1) * sizeof(T));
}
}  // namespace

namespace {
int create_impl(bta_ctx* c, const bta_model_desc* desc, const bta_obs* obs);
}

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
  DeviceGuard guard(device);
  bta_ctx* c = new bta_ctx();   // value-initialised: every pointer / handle starts as null, so bta_destroy is safe
  c->device = device;
  const int rc = create_impl(c, desc, obs);
  if (rc != BTA_OK) {
    bta_destroy(c);             // releases whatever had been allocated before the failure
    return rc;
  }
  *out = c;
  return BTA_OK;
}

namespace {
int create_impl(bta_ctx* c, const bta_model_desc* desc, const bta_obs* obs) {
  const int device = c->device;
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
  c->m = obs->m;
  c->launches = 0;
  c->last_pivot = 0;
  c->have_x = false;
  const long long m = obs->m;
  for (long long i = 0; i < m; ++i) {
    if (obs->var[i] < 0 || obs->var[i] >= md.k || obs->node[i] < 0 || obs->node[i] >= md.ns || obs->time[i] < 0 ||
        obs->time[i] >= md.nt) {
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
  BTA_CUDA_OK(dev_alloc(&c->x_keep, (size_t)md.N));
  SmallLayout L = small_layout(md);
  c->small_doubles = L.total;
  BTA_CUDA_OK(dev_alloc(&c->small, L.total));
  BTA_CUDA_OK(cudaMemset(c->small, 0, L.total * sizeof(double)));
  BTA_CUDA_OK(cudaMallocHost((void**)&c->host_pinned, 4096 * sizeof(double)));
  // The four chains run at equal (lowest) priority: with four chains in flight the GPU is throughput-bound, and
  // prioritising whole chains only moves time between them (measured in round 1).  Only the small latency-bound
  // kernels of every chain get a high-priority companion stream (s_hi below).
  int prio_lo = 0, prio_hi = 0;
  BTA_CUDA_OK(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
  BTA_CUDA_OK(cudaStreamCreateWithPriority(&c->s_main, cudaStreamNonBlocking, prio_lo));
  BTA_CUDA_OK(cudaStreamCreateWithPriority(&c->s_aux[0], cudaStreamNonBlocking, prio_lo));
  BTA_CUDA_OK(cudaStreamCreateWithPriority(&c->s_side, cudaStreamNonBlocking, prio_lo));
  BTA_CUDA_OK(cudaStreamCreateWithPriority(&c->s_aux[1], cudaStreamNonBlocking, prio_lo));
  for (int q = 0; q < 2; ++q) {
    c->graph_exec[q] = nullptr;
    c->graph_ws[q] = nullptr;
    c->graph_launches[q] = 0;
  }
  c->grad_calls = 0;
  c->trace_on = getenv("BTA_TRACE") != nullptr;
  {
    auto env = [](const char* name, int dflt) {
      const char* e = getenv(name);
      return e ? atoi(e) : dflt;
    };
    c->opt.twist = env("BTA_TWIST", c->opt.twist);
    c->opt.lanes = env("BTA_LANES", c->opt.lanes);
    c->opt.split = env("BTA_SPLIT", c->opt.split);
    c->opt.graph = env("BTA_GRAPH", c->opt.graph);
    c->opt.serial = env("BTA_SERIAL_CHAINS", c->opt.serial);
    c->opt.pipeline = env("BTA_PIPELINE", c->opt.pipeline);
    c->opt.partitions = env("BTA_PARTITIONS", c->opt.partitions);
    c->opt.rows = env("BTA_ROWS", c->opt.rows);
    g_tile_thresh = env("BTA_TILE_THRESH", (int)g_tile_thresh);
    g_tile_waves = env("BTA_TILE_WAVES", g_tile_waves);
    g_pdl = env("BTA_PDL", g_pdl);
  }
  c->store_mode = BTA_STORE_FACTOR;
  for (auto& e : c->ev) BTA_CUDA_OK(cudaEventCreate(&e));
  for (auto& q : c->s_hi) BTA_CUDA_OK(cudaStreamCreateWithPriority(&q, cudaStreamNonBlocking, prio_hi));
  for (auto& q : c->s_x) BTA_CUDA_OK(cudaStreamCreateWithPriority(&q, cudaStreamNonBlocking, prio_lo));
  for (auto& q : c->s_r) BTA_CUDA_OK(cudaStreamCreateWithPriority(&q, cudaStreamNonBlocking, prio_hi));
  for (auto& q : c->s_g) BTA_CUDA_OK(cudaStreamCreateWithPriority(&q, cudaStreamNonBlocking, prio_lo));
  for (auto& e : c->ev_sw) BTA_CUDA_OK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  for (auto& q : c->s_copy) BTA_CUDA_OK(cudaStreamCreateWithPriority(&q, cudaStreamNonBlocking, prio_lo));
  for (auto& q : c->ev_ring)
    for (auto& e : q) BTA_CUDA_OK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  for (auto& q : c->ev_pipe)
    for (auto& e : q) BTA_CUDA_OK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  c->ev_sw_next = 0;
  if (m > 0) {
    BTA_CUDA_OK(cudaMemcpy(c->o_var, obs->var, m * sizeof(int), cudaMemcpyHostToDevice));
    BTA_CUDA_OK(cudaMemcpy(c->o_node, obs->node, m * sizeof(int), cudaMemcpyHostToDevice));
    BTA_CUDA_OK(cudaMemcpy(c->o_time, obs->time, m * sizeof(int), cudaMemcpyHostToDevice));
    BTA_CUDA_OK(cudaMemcpy(c->o_cov, obs->cov, m * md.apr * sizeof(double), cudaMemcpyHostToDevice));
    BTA_CUDA_OK(cudaMemcpy(c->o_y, obs->y, m * sizeof(double), cudaMemcpyHostToDevice));
  }
  BTA_CUDA_OK(run_setup_aggregates(c, 0));
  (void)device;
  return BTA_OK;
}
}  // namespace

extern "C" int bta_destroy(bta_ctx* c) {
  if (!c) return BTA_OK;
  DeviceGuard guard(c->device);
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
  cudaFree(c->x_keep);
  if (c->host_pinned) cudaFreeHost(c->host_pinned);
  for (int q = 0; q < 2; ++q)
    if (c->graph_exec[q]) cudaGraphExecDestroy(c->graph_exec[q]);
  auto kill_stream = [](cudaStream_t q) {
    if (q) cudaStreamDestroy(q);
  };
  auto kill_event = [](cudaEvent_t e) {
    if (e) cudaEventDestroy(e);
  };
  kill_stream(c->s_side);
  kill_stream(c->s_main);
  for (auto& q : c->s_aux) kill_stream(q);
  for (auto& q : c->s_hi) kill_stream(q);
  for (auto& q : c->s_x) kill_stream(q);
  for (auto& q : c->s_r) kill_stream(q);
  for (auto& q : c->s_g) kill_stream(q);
  for (auto& q : c->s_copy) kill_stream(q);
  for (int m = 0; m < 2; ++m)
    for (int p = 0; p < 8; ++p) {
      kill_stream(c->s_part[m][p]);
      kill_stream(c->s_part_hi[m][p]);
      kill_stream(c->s_part_x[m][p]);
      kill_stream(c->s_part_r[m][p]);
    }
  for (auto& q : c->ev_ring)
    for (auto& e : q) kill_event(e);
  for (auto& e : c->ev) kill_event(e);
  for (auto& e : c->ev_sw) kill_event(e);
  for (auto& q : c->ev_pipe)
    for (auto& e : q) kill_event(e);
  delete c;
  return BTA_OK;
}

extern "C" int32_t bta_num_hyper(const bta_ctx* c) { return c ? c->md.d : 0; }
extern "C" int64_t bta_latent_size(const bta_ctx* c) { return c ? c->md.N : 0; }
extern "C" int64_t bta_last_pivot(const bta_ctx* c) { return c ? c->last_pivot : 0; }
extern "C" int64_t bta_kernel_launches(const bta_ctx* c) { return c ? c->launches : 0; }

extern "C" int bta_set_store_mode(bta_ctx* c, int mode) {
  if (!c || (mode != BTA_STORE_FACTOR && mode != BTA_STORE_CARRY && mode != BTA_STORE_HOST)) {
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

extern "C" size_t bta_host_bytes(const bta_ctx* c) {
  if (!c || c->md.nt < 3) return 0;
  return (size_t)2 * (size_t)(c->md.nt - 1) * (size_t)c->md.b * (size_t)c->md.b * sizeof(double);
}
extern "C" int bta_set_host_buffer(bta_ctx* c, void* host, size_t bytes) {
  if (!c || (host && bytes < bta_host_bytes(c))) {
    bta_set_error("bta_set_host_buffer: null ctx, or fewer than bta_host_bytes(ctx) bytes");
    return BTA_ERR_ARG;
  }
  for (int q = 0; q < 2; ++q)
    if (c->graph_exec[q]) {  // a cached graph holds the old host pointers
      cudaGraphExecDestroy(c->graph_exec[q]);
      c->graph_exec[q] = nullptr;
    }
  c->host_buf = (double*)host;
  c->host_bytes = host ? bytes : 0;
  return BTA_OK;
}

namespace {
int* option_slot(bta_ctx* c, int option) {
  switch (option) {
    case BTA_OPT_TWIST: return &c->opt.twist;
    case BTA_OPT_LANES: return &c->opt.lanes;
    case BTA_OPT_SPLIT: return &c->opt.split;
    case BTA_OPT_GRAPH: return &c->opt.graph;
    case BTA_OPT_SERIAL: return &c->opt.serial;
    case BTA_OPT_PIPELINE: return &c->opt.pipeline;
    case BTA_OPT_PARTITIONS: return &c->opt.partitions;
    case BTA_OPT_ROWS: return &c->opt.rows;
  }
  return nullptr;
}
}  // namespace

extern "C" int bta_set_option(bta_ctx* c, int option, int value) {
  if (option == BTA_OPT_TILE_THRESH || option == BTA_OPT_TILE_WAVES || option == BTA_OPT_PDL) {  // process-global
    if (option == BTA_OPT_TILE_THRESH) g_tile_thresh = value;
    else if (option == BTA_OPT_TILE_WAVES) g_tile_waves = value;
    else g_pdl = value;
    if (c)
      for (int q = 0; q < 2; ++q)
        if (c->graph_exec[q]) {
          cudaGraphExecDestroy(c->graph_exec[q]);
          c->graph_exec[q] = nullptr;
        }
    return BTA_OK;
  }
  int* slot = c ? option_slot(c, option) : nullptr;
  if (!slot) {
    bta_set_error("bta_set_option: null ctx or unknown option");
    return BTA_ERR_ARG;
  }
  if (*slot != value)
    for (int q = 0; q < 2; ++q)
      if (c->graph_exec[q]) {  // a cached graph was captured with the other setting
        cudaGraphExecDestroy(c->graph_exec[q]);
        c->graph_exec[q] = nullptr;
      }
  *slot = value;
  return BTA_OK;
}
extern "C" int bta_get_option(const bta_ctx* c, int option) {
  int* slot = c ? option_slot(const_cast<bta_ctx*>(c), option) : nullptr;
  return slot ? *slot : -1;
}
