// Small helpers shared by the entry-point files (api.cu, partition.cu).
#pragma once
#include "sweep.h"

struct Bump {  // carves the caller's workspace into 256-byte aligned pieces (base = nullptr: size query)
  char* base;
  size_t off = 0;
  explicit Bump(void* p) : base((char*)p) {}
  double* take(size_t doubles) {
    double* r = (double*)(base + off);
    off += (doubles * sizeof(double) + 255) / 256 * 256;
    return r;
  }
};

inline int bad(const char* msg) {
  bta_set_error(msg);
  return BTA_ERR_ARG;
}

// partition.cu -- time-domain partitioning with P partitions and a reduced system
constexpr int BTA_PMAX = 8;
bool use_partitions(const bta_ctx* c);              // opt.partitions >= 2 and the model is long enough
size_t part_ws_bytes(const bta_ctx* c);
int enqueue_gradient_partitioned(bta_ctx* c, void* ws, cudaStream_t s0, bool timed, bool value_only);
