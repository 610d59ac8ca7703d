// mkf_scan.cuh — exclusive prefix sum of unsigned counts (reduce / scan-of-partials / downsweep), used by the
// hit index (a1) and by duplicate removal (a10). After the call `cnt` holds the same offsets as `out`
// (ready to be used as scatter cursors) and out[n] = total.
#pragma once
#include "mkf_ctx.h"

namespace mkf {

constexpr int SCAN_BLOCK = 256, SCAN_ITEMS = 8, SCAN_TILE = SCAN_BLOCK * SCAN_ITEMS;
constexpr unsigned SCAN_TOTAL_UNKNOWN = 0xffffffffu;    // as `total` of exclusive_scan_u32: out[n] = the sum of the counts

static __device__ __forceinline__ unsigned block_exclusive_scan(unsigned v, unsigned* total) {   // SCAN_BLOCK threads
  __shared__ unsigned s_w[SCAN_BLOCK / 32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  unsigned inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
  if (lane == 31) s_w[w] = inc;
  __syncthreads();
  if (w == 0) {
    unsigned x = lane < SCAN_BLOCK / 32 ? s_w[lane] : 0u, xi = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, xi, o); if (lane >= o) xi += t; }
    if (lane < SCAN_BLOCK / 32) s_w[lane] = xi - x;
    if (lane == 31) *total = xi;
  }
  __syncthreads();
  const unsigned r = s_w[w] + inc - v;
  __syncthreads();
  return r;
}

static __global__ void __launch_bounds__(SCAN_BLOCK) scan_reduce(const unsigned* __restrict__ cnt, size_t n, unsigned* partial) {
  const size_t base = (size_t)blockIdx.x * SCAN_TILE;
  unsigned s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; k++) { const size_t i = base + (size_t)k * SCAN_BLOCK + threadIdx.x; if (i < n) s += cnt[i]; }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  __shared__ unsigned s_w[SCAN_BLOCK / 32];
  if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) { unsigned t = 0; for (int w = 0; w < SCAN_BLOCK / 32; w++) t += s_w[w]; partial[blockIdx.x] = t; }
}

// single CTA: exclusive scan of the tile sums, in place
static __global__ void __launch_bounds__(SCAN_BLOCK) scan_partials(unsigned* partial, int np) {
  __shared__ unsigned s_total;
  unsigned carry = 0;
  for (int base = 0; base < np; base += SCAN_BLOCK) {
    const int i = base + threadIdx.x;
    const unsigned v = i < np ? partial[i] : 0u;
    const unsigned ex = block_exclusive_scan(v, &s_total);
    if (i < np) partial[i] = carry + ex;
    carry += s_total;
    __syncthreads();
  }
}

// exclusive scan inside each tile + tile offset -> bin_off; the counts are replaced by the same offsets (cursors)
static __global__ void __launch_bounds__(SCAN_BLOCK) scan_down(unsigned* cnt, size_t n, const unsigned* __restrict__ partial,
                                                           unsigned* bin_off, unsigned total_hits) {
  __shared__ unsigned s_total;
  const size_t base = (size_t)blockIdx.x * SCAN_TILE + (size_t)threadIdx.x * SCAN_ITEMS;   // blocked arrangement
  unsigned v[SCAN_ITEMS], s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; k++) { v[k] = base + k < n ? cnt[base + k] : 0u; s += v[k]; }
  unsigned run = partial[blockIdx.x] + block_exclusive_scan(s, &s_total);
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; k++) {
    if (base + k < n) { bin_off[base + k] = run; cnt[base + k] = run; }
    run += v[k];
    if (total_hits == SCAN_TOTAL_UNKNOWN && base + k == n - 1) bin_off[n] = run;       // the sum itself
  }
  if (total_hits != SCAN_TOTAL_UNKNOWN && blockIdx.x == 0 && threadIdx.x == 0) bin_off[n] = total_hits;
}

inline size_t scan_partial_bytes(size_t n) { return align256(((n + SCAN_TILE - 1) / SCAN_TILE + 1) * 4); }

static inline int exclusive_scan_u32(mkf_ctx* c, unsigned* cnt, size_t n, unsigned* partial, unsigned* out, unsigned total,
                                     cudaStream_t st) {
  const size_t ntiles = (n + SCAN_TILE - 1) / SCAN_TILE;
  if (ntiles == 0 || ntiles > 0x7fffffffu) return fail(c, MKF_UNSUPPORTED, "exclusive_scan: size out of range");
  scan_reduce<<<(unsigned)ntiles, SCAN_BLOCK, 0, st>>>(cnt, n, partial);
  MKF_LAUNCHED(c, "scan_reduce");
  scan_partials<<<1, SCAN_BLOCK, 0, st>>>(partial, (int)ntiles);
  MKF_LAUNCHED(c, "scan_partials");
  scan_down<<<(unsigned)ntiles, SCAN_BLOCK, 0, st>>>(cnt, n, partial, out, total);
  MKF_LAUNCHED(c, "scan_down");
  return MKF_OK;
}

}  // namespace mkf
