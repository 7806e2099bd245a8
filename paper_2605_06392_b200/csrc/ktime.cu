// Per-kernel-class timing (include/bta_diag.h: bta_diag_ktime_begin / _end): while armed, every kernel launcher of the
// library brackets its launch with a pair of CUDA events on the launching stream and registers the algorithmic flops and
// bytes of that launch.  Meant for one step with BTA_OPT_SERIAL = 1 (one stream: the intervals are exclusive and add up
// to the step); bench.py derives from it the in-step rate of the dominant kernel, its share of the step and the achieved
// GB/s of the bandwidth-bound classes.  Not armed: one predictable branch per launch.
#include <mutex>

#include "common.cuh"

bool g_ktime_on = false;

namespace {
struct Rec {
  cudaEvent_t e0, e1;
  int cls;
  double flop, bytes;
};
std::vector<Rec> g_recs;
std::vector<cudaEvent_t> g_free;
std::mutex g_mu;

cudaEvent_t take_event() {
  if (!g_free.empty()) {
    cudaEvent_t e = g_free.back();
    g_free.pop_back();
    return e;
  }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}
}  // namespace

KTimeScope::KTimeScope(int cls, cudaStream_t st, double flop, double bytes) : idx(-1), stream(st) {
  if (!g_ktime_on) return;
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) return;
  std::lock_guard<std::mutex> lk(g_mu);
  Rec r{take_event(), take_event(), cls, flop, bytes};
  if (!r.e0 || !r.e1) return;
  cudaEventRecord(r.e0, st);
  idx = (long long)g_recs.size();
  g_recs.push_back(r);
}
KTimeScope::~KTimeScope() {
  if (idx < 0) return;
  std::lock_guard<std::mutex> lk(g_mu);
  cudaEventRecord(g_recs[(size_t)idx].e1, stream);
}

extern "C" int bta_diag_ktime_begin(void) {
  std::lock_guard<std::mutex> lk(g_mu);
  for (auto& r : g_recs) {
    g_free.push_back(r.e0);
    g_free.push_back(r.e1);
  }
  g_recs.clear();
  g_ktime_on = true;
  return BTA_OK;
}

extern "C" int bta_diag_ktime_end(double* ms, double* flop, double* bytes, long long* count) {
  BTA_CUDA_OK(cudaDeviceSynchronize());
  std::lock_guard<std::mutex> lk(g_mu);
  g_ktime_on = false;
  for (int q = 0; q < BTA_KC_COUNT; ++q) {
    if (ms) ms[q] = 0.0;
    if (flop) flop[q] = 0.0;
    if (bytes) bytes[q] = 0.0;
    if (count) count[q] = 0;
  }
  for (auto& r : g_recs) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, r.e0, r.e1) != cudaSuccess) t = 0.f;
    if (ms) ms[r.cls] += t;
    if (flop) flop[r.cls] += r.flop;
    if (bytes) bytes[r.cls] += r.bytes;
    if (count) count[r.cls] += 1;
    g_free.push_back(r.e0);
    g_free.push_back(r.e1);
  }
  g_recs.clear();
  return BTA_OK;
}
