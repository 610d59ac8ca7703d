// mkf_ctx.h — host-side context shared by the translation units of libmkf.so.
#pragma once
#include <cuda_runtime.h>
#include <cstdio>
#include <cstring>
#include "../../include/mkf.h"
#include "mkf_dev.cuh"

// State of the host-buffer entry points (mkf_host.cu): a grow-only device arena, three streams (copy in, kernels,
// copy out) and a pool of events, all created at the first host call and kept until mkf_destroy, so that repeated
// calls allocate nothing ("a memory pool to pay the allocation overhead only at the beginning and end of job").
struct mkf_host_state {
  char* base = nullptr; size_t cap = 0;
  cudaStream_t s_in = nullptr, s_k = nullptr, s_out = nullptr;
  cudaEvent_t ev[128] = {};
  int n_ev = 0;
};

struct mkf_ctx {
  mkf::GeomDev g;
  mkf::ParamsDev p;
  int max_plan_len;
  long long launches;
  char err[256];
  mkf_host_state* host;
  unsigned long long* build_counters;      // device, or null (mkf_set_build_counters)
};

namespace mkf {
inline int fail(mkf_ctx* c, int code, const char* what) {
  if (c) snprintf(c->err, sizeof(c->err), "%s", what);
  return code;
}
inline int cuda_fail(mkf_ctx* c, cudaError_t e, const char* where) {
  if (c) snprintf(c->err, sizeof(c->err), "%s: %s", where, cudaGetErrorString(e));
  return MKF_CUDA_ERROR;
}
// after a kernel launch: count it and pick up launch-configuration errors (no synchronisation)
#define MKF_LAUNCHED(ctx, name)                                        \
  do {                                                                 \
    (ctx)->launches++;                                                 \
    cudaError_t e__ = cudaGetLastError();                              \
    if (e__ != cudaSuccess) return mkf::cuda_fail((ctx), e__, name);   \
  } while (0)
inline size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }
inline HitsDev hits_dev(const mkf_hits* h) {
  HitsDev d; d.n_events = h->n_events; d.n_hits = h->n_hits; d.layer_off = h->layer_off;
  d.x = h->x; d.y = h->y; d.z = h->z; d.V = h->V; d.rec = (const float4*)h->rec; d.module = h->module; return d;
}
}  // namespace mkf
