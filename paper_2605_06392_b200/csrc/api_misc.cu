// Error text, and the thin measurement entry point bta_gemm of include/bta_diag.h.
#include "common.cuh"

static thread_local std::string g_err;

void bta_set_error(const char* msg) { g_err = msg; }
void bta_set_error_cuda(cudaError_t e, const char* what, const char* file, int line) {
  char buf[512];
  snprintf(buf, sizeof buf, "CUDA error %d (%s) in %s at %s:%d", (int)e, cudaGetErrorString(e), what, file, line);
  g_err = buf;
}
extern "C" const char* bta_last_error(void) { return g_err.c_str(); }

extern "C" int bta_gemm(int mode, int M, int N, int K, double alpha, const double* A, int lda, const double* B,
                        int ldb, double beta, double* C, int ldc, int klo, int khi, int out, void* stream) {
  if (mode < 0 || mode > 2 || M < 0 || N < 0 || K < 0) {
    bta_set_error("bta_gemm: bad mode or size");
    return BTA_ERR_ARG;
  }
  GemmArgs g{A, B, C, M, N, K, lda, ldb, ldc, alpha, beta, mode, klo, khi, out, nullptr, 0, 0};
  BTA_CUDA_OK(launch_gemm(g, (cudaStream_t)stream));
  return BTA_OK;
}
