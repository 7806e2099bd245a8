// FP64 ceiling microbenchmarks (bench.py's roofline denominators): register-resident issue loops on every
// SM, no memory traffic.  kind 0: mma.sync.m8n8k4.f64 (DMMA.8x8x4);  kind 1: DFMA.
#include "common.cuh"

namespace {

template <int NACC>
__global__ void __launch_bounds__(256) dmma_loop(int iters, double* sink) {
  double c[NACC][2];
#pragma unroll
  for (int i = 0; i < NACC; ++i) c[i][0] = c[i][1] = 0.0;
  double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < NACC; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                   : "+d"(c[i][0]), "+d"(c[i][1])
                   : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < NACC; ++i) s += c[i][0] + c[i][1];
  if (s == 123.456) sink[0] = s;
}

template <int NACC>
__global__ void __launch_bounds__(256) dfma_loop(int iters, double* sink) {
  double c[NACC];
#pragma unroll
  for (int i = 0; i < NACC; ++i) c[i] = i;
  double a = 1.0 + threadIdx.x * 1e-9, b = 1e-9 * threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < NACC; ++i) c[i] = fma(c[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < NACC; ++i) s += c[i];
  if (s == 123.456) sink[0] = s;
}

}  // namespace

extern "C" int bta_fp64_peak(int kind, int iters, double* tflops, double* ms_out, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  BTA_CUDA_OK(cudaGetDevice(&dev));
  BTA_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  double* sink = nullptr;
  BTA_CUDA_OK(cudaMalloc(&sink, 8));
  cudaEvent_t e0, e1;
  BTA_CUDA_OK(cudaEventCreate(&e0));
  BTA_CUDA_OK(cudaEventCreate(&e1));
  constexpr int NACC = 16;
  const int ctas = sms, threads = 256;  // 8 warps/SM: measured best (more resident warps lower the DMMA rate)
  for (int rep = 0; rep < 2; ++rep) {  // first pass warms up
    BTA_CUDA_OK(cudaEventRecord(e0, st));
    if (kind == 0)
      dmma_loop<NACC><<<ctas, threads, 0, st>>>(iters, sink);
    else
      dfma_loop<NACC><<<ctas, threads, 0, st>>>(iters, sink);
    BTA_CUDA_OK(cudaGetLastError());
    BTA_CUDA_OK(cudaEventRecord(e1, st));
    BTA_CUDA_OK(cudaEventSynchronize(e1));
  }
  float ms = 0.f;
  BTA_CUDA_OK(cudaEventElapsedTime(&ms, e0, e1));
  double flop = kind == 0 ? (double)ctas * (threads / 32) * (double)iters * NACC * 512.0
                          : (double)ctas * threads * (double)iters * NACC * 2.0;
  if (tflops) *tflops = flop / (ms * 1e-3) / 1e12;
  if (ms_out) *ms_out = ms;
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  return BTA_OK;
}
