// mkf_dedup.cu — a10 / C10: duplicate removal ("duplicate tracks ... explicitly removed in an
// additional processing step"). Integer-only: must agree with the oracle exactly.
//
// Pairwise dominance (U15): track i is removed iff some j != i of the same event shares more than
// dup_frac * min(nhits_i, nhits_j) hits with it and ranks higher (score, then lower index).
// Only tracks that share at least one hit can dominate each other, so an inverted index hit -> tracks is built
// (count / scan / fill) and each track looks only at the tracks listed under its own hits.
#include "mkf_ctx.h"
#include "mkf_scan.cuh"

using namespace mkf;

namespace {

constexpr int DD_BLOCK = 256;

struct DdArgs {
  int n_events, n, n_hits, mpl; const int* track_off; const int* hit_ids; const int* nhits; const float* score;
  unsigned* cnt; unsigned* off; int* list; unsigned char* keep; int* n_kept; float dup_frac;
};

__global__ void __launch_bounds__(DD_BLOCK) dd_count(const __grid_constant__ DdArgs a) {
  const size_t k = (size_t)blockIdx.x * DD_BLOCK + threadIdx.x;
  if (k >= (size_t)a.n * a.mpl) return;
  const int h = a.hit_ids[k];
  if (h >= 0 && h < a.n_hits) atomicAdd(&a.cnt[h], 1u);
}

__global__ void __launch_bounds__(DD_BLOCK) dd_fill(const __grid_constant__ DdArgs a) {
  const size_t k = (size_t)blockIdx.x * DD_BLOCK + threadIdx.x;
  if (k >= (size_t)a.n * a.mpl) return;
  const int h = a.hit_ids[k];
  if (h >= 0 && h < a.n_hits) a.list[atomicAdd(&a.cnt[h], 1u)] = (int)(k % (size_t)a.n);
}

// |ids_i ∩ ids_j| (entries of j that are hits of i) is the number of times j appears in the lists filed under the
// DISTINCT hits of i, so one warp per track gathers those lists into shared memory and counts multiplicities: with at
// most 32 entries one match.any does it. Tracks whose lists hold more than DD_CAP entries, and plans longer than a
// warp, take the plain loop (lane 0).
constexpr int DD_CAP = 128, DD_WARPS = DD_BLOCK / 32;

__device__ bool dd_dominated_slow(const DdArgs& a, int i, int eb, int ee) {
  const size_t n = (size_t)a.n;
  const int nhi = a.nhits[i];
  const float si = a.score[i];
  for (int s = 0; s < a.mpl; s++) {
    const int h = a.hit_ids[(size_t)s * n + i];
    if (h < 0 || h >= a.n_hits) continue;
    for (unsigned t = a.off[h]; t < a.off[h + 1]; t++) {
      const int j = a.list[t];
      if (j == i || j < eb || j >= ee) continue;
      const float sj = a.score[j];
      if (!(sj > si || (sj == si && j < i))) continue;       // j must rank higher
      const int mn = min(nhi, a.nhits[j]);
      if (mn <= 0) continue;
      int shared = 0;                                         // |ids_i ∩ ids_j|
      for (int c = 0; c < a.mpl; c++) {
        const int hc = a.hit_ids[(size_t)c * n + j];
        if (hc < 0) continue;
        for (int d = 0; d < a.mpl; d++) if (a.hit_ids[(size_t)d * n + i] == hc) { shared++; break; }
      }
      if ((double)shared > (double)a.dup_frac * (double)mn) return true;
    }
  }
  return false;
}

__global__ void __launch_bounds__(DD_BLOCK) dd_mark(const __grid_constant__ DdArgs a) {
  __shared__ int s_e[DD_WARPS][DD_CAP];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int i = blockIdx.x * DD_WARPS + w;
  if (i >= a.n) return;                                       // whole warp
  int* E = s_e[w];
  // event of track i: last ev with track_off[ev] <= i
  int lo = 0, hi = a.n_events;
  while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (a.track_off[mid] <= i) lo = mid; else hi = mid; }
  const int eb = a.track_off[lo], ee = a.track_off[lo + 1];
  const size_t n = (size_t)a.n;
  int total = 0;
  for (int s0 = 0; s0 < a.mpl; s0 += 32) {
    const int s = s0 + lane;
    int h = -1;
    if (s < a.mpl) h = a.hit_ids[(size_t)s * n + i];
    unsigned b = 0; int len = 0;
    const bool valid = h >= 0 && h < a.n_hits;
    const unsigned same = __match_any_sync(0xffffffffu, valid ? h : -1 - lane);
    if (valid && (__ffs(same) - 1) == lane) { b = a.off[h]; len = (int)(a.off[h + 1] - b); }       // first occurrence of h in i
    int inc = len;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int t2 = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t2; }
    const int pos = total + inc - len;
    for (int k = 0; k < len; k++) if (pos + k < DD_CAP) E[pos + k] = a.list[b + k];
    total += __shfl_sync(0xffffffffu, inc, 31);
  }
  __syncwarp();
  bool removed = false;
  if (total > DD_CAP || a.mpl > 32) { if (lane == 0) removed = dd_dominated_slow(a, i, eb, ee); }
  else {
    const int nhi = a.nhits[i];
    const float si = a.score[i];
    for (int e0 = 0; e0 < total; e0 += 32) {
      const int e = e0 + lane;
      const int j = e < total ? E[e] : -1 - lane;
      int m; bool first;
      if (total <= 32) {
        const unsigned mm = __match_any_sync(0xffffffffu, j);
        m = __popc(mm); first = (__ffs(mm) - 1) == lane;
      } else {
        m = 0; first = true;
        for (int q = 0; q < total; q++) { const bool eq = E[q] == j; m += eq; if (eq && q < e) first = false; }
      }
      if (e < total && first && j != i && j >= eb && j < ee) {
        const float sj = a.score[j];
        if (sj > si || (sj == si && j < i)) {                 // j ranks higher
          const int mn = min(nhi, a.nhits[j]);
          if (mn > 0 && (double)m > (double)a.dup_frac * (double)mn) removed = true;
        }
      }
    }
  }
  removed = __any_sync(0xffffffffu, removed);
  if (lane == 0) a.keep[i] = removed ? 0 : 1;
}

__global__ void __launch_bounds__(DD_BLOCK) dd_count_kept(const __grid_constant__ DdArgs a) {
  const int ev = blockIdx.x;
  const int b = a.track_off[ev], e = a.track_off[ev + 1];
  int s = 0;
  for (int i = b + threadIdx.x; i < e; i += DD_BLOCK) s += a.keep[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  __shared__ int s_w[DD_BLOCK / 32];
  if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) { int t = 0; for (int w = 0; w < DD_BLOCK / 32; w++) t += s_w[w]; a.n_kept[ev] = t; }
}

}  // namespace

namespace mkf {
size_t dedup_ws_bytes(int n_hits, int n, int mpl) {
  return align256(((size_t)n_hits + 2) * 4) * 2 + scan_partial_bytes((size_t)n_hits + 1) + align256((size_t)n * mpl * 4);
}
}  // namespace mkf

extern "C" int mkf_remove_duplicates(mkf_ctx* c, int n_events, int n, int n_hits, const int* track_off, const int* hit_ids,
                                     int max_plan_len, const int* nhits, const float* score, unsigned char* keep,
                                     int* n_kept, void* ws, size_t ws_bytes, void* stream) {
  if (!c) return MKF_INVALID_ARG;
  if (!track_off || !hit_ids || !nhits || !score || !keep || !n_kept) return fail(c, MKF_INVALID_ARG, "mkf_remove_duplicates: null argument");
  if (n_events < 1 || n < 0 || n_hits < 0 || max_plan_len < 1) return fail(c, MKF_INVALID_ARG, "mkf_remove_duplicates: bad sizes");
  const size_t need = dedup_ws_bytes(n_hits, n, max_plan_len);
  if (ws_bytes < need || !ws) return fail(c, MKF_WORKSPACE_TOO_SMALL, "mkf_remove_duplicates: workspace too small");
  cudaStream_t st = (cudaStream_t)stream;
  char* w = (char*)ws;
  DdArgs a;
  a.n_events = n_events; a.n = n; a.n_hits = n_hits; a.mpl = max_plan_len; a.track_off = track_off; a.hit_ids = hit_ids;
  a.nhits = nhits; a.score = score; a.keep = keep; a.n_kept = n_kept; a.dup_frac = c->p.dup_frac;
  a.cnt = (unsigned*)w; w += align256(((size_t)n_hits + 2) * 4);
  a.off = (unsigned*)w; w += align256(((size_t)n_hits + 2) * 4);
  unsigned* partial = (unsigned*)w; w += scan_partial_bytes((size_t)n_hits + 1);
  a.list = (int*)w;
  cudaError_t e = cudaMemsetAsync(a.cnt, 0, ((size_t)n_hits + 1) * 4, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "mkf_remove_duplicates: memset");
  const size_t total = (size_t)n * max_plan_len;
  if (total > 0) {
    const unsigned grid = (unsigned)((total + DD_BLOCK - 1) / DD_BLOCK);
    dd_count<<<grid, DD_BLOCK, 0, st>>>(a);
    MKF_LAUNCHED(c, "dd_count");
    // the trailing total (off[n_hits]) is the sum itself: scan n_hits+1 counts whose last one is zero
    { const int rc = exclusive_scan_u32(c, a.cnt, (size_t)n_hits + 1, partial, a.off, 0u, st); if (rc) return rc; }
    dd_fill<<<grid, DD_BLOCK, 0, st>>>(a);
    MKF_LAUNCHED(c, "dd_fill");
    dd_mark<<<(n + DD_WARPS - 1) / DD_WARPS, DD_BLOCK, 0, st>>>(a);
    MKF_LAUNCHED(c, "dd_mark");
  }
  dd_count_kept<<<n_events, DD_BLOCK, 0, st>>>(a);
  MKF_LAUNCHED(c, "dd_count_kept");
  return MKF_OK;
}
