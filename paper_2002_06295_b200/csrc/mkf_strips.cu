// mkf_strips.cu — strip clustering (reading R8 of DESIGN.md) in ONE pass over the strips.
//
// HBM-bound: 7 bytes per strip in (adc u16, noise f32, bad u8), 20 bytes per kept cluster out. One CTA takes a tile
// of SC_TILE consecutive strips of the concatenated batch (tiles are handed out by a ticket so that a tile's
// predecessors are always resident), each thread 8 consecutive strips with 16-byte loads:
//   1. threshold bits (pass / bad) of the tile and of a 32-strip halo to its left, module-start bits from module_off;
//   2. a passing strip starts a cluster iff no passing strip of its module lies within the allowed gap to its left
//      (bit tests on a 40-strip window per thread);
//   3. the thread that owns a start walks its cluster in strip order (the sums of R8 are order-dependent in fp64)
//      and stages the record in shared memory;
//   4. the number of kept clusters of the tile goes through a decoupled look-back scan over the tiles, and the
//      staged records are written compacted, in (module, first strip) order.
// Nothing here is shared with oracle/.
#include "mkf_ctx.h"
#include <cstdint>

namespace mkf {

constexpr int SC_THREADS = 256, SC_PER = 8, SC_TILE = SC_THREADS * SC_PER, SC_HALO = 32;
constexpr int SC_MS_WORDS = (SC_TILE + SC_HALO) / 32;

struct ScArgs {
  int n_modules, n_strips, n_tiles;
  const int* moff; const unsigned short* adc; const float* noise; const unsigned char* bad;
  float seed_thr, chan_thr, clus_thr; int min_charge, max_holes, max_bad;
  int cap; int *o_module, *o_first, *o_last; unsigned* o_charge; float* o_bary; int* n_clusters;
  unsigned long long* tile_state;       // [n_tiles]: flag << 32 | value; flag 1 = tile aggregate, 2 = inclusive prefix
  unsigned* ticket;
};

// largest m in [lo, hi) with moff[m] <= g (moff ascending; hi > lo and moff[lo] <= g)
__device__ __forceinline__ int module_of(const int* __restrict__ moff, int lo, int hi, int g) {
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(moff + mid) <= g) lo = mid; else hi = mid;
  }
  return lo;
}

// threshold bits of 8 consecutive strips starting at g0 (multiple of 8): bit k of pass / bad
__device__ __forceinline__ void strip_bits(const ScArgs& a, int g0, unsigned& pass, unsigned& bad) {
  pass = 0; bad = 0;
  if (g0 + SC_PER <= a.n_strips) {
    const uint4 av = __ldg(reinterpret_cast<const uint4*>(a.adc + g0));
    const float4 n0 = __ldg(reinterpret_cast<const float4*>(a.noise + g0));
    const float4 n1 = __ldg(reinterpret_cast<const float4*>(a.noise + g0) + 1);
    const uint2 bv = __ldg(reinterpret_cast<const uint2*>(a.bad + g0));
    const unsigned aw[4] = {av.x, av.y, av.z, av.w};
    const float nz[8] = {n0.x, n0.y, n0.z, n0.w, n1.x, n1.y, n1.z, n1.w};
#pragma unroll
    for (int k = 0; k < 8; k++) {
      const unsigned adc = (aw[k >> 1] >> ((k & 1) * 16)) & 0xffffu;
      const unsigned b = (((k < 4 ? bv.x : bv.y) >> ((k & 3) * 8)) & 0xffu) != 0;
      bad |= b << k;
      pass |= (unsigned)(!b && (float)adc > a.chan_thr * nz[k]) << k;
    }
  } else {
    for (int k = 0; k < 8 && g0 + k < a.n_strips; k++) {
      const unsigned b = a.bad[g0 + k] != 0;
      bad |= b << k;
      pass |= (unsigned)(!b && (float)a.adc[g0 + k] > a.chan_thr * a.noise[g0 + k]) << k;
    }
  }
}

__global__ void __launch_bounds__(SC_THREADS) sc_cluster_kernel(const ScArgs a) {
  __shared__ unsigned char s_pass[SC_THREADS + 4], s_bad[SC_THREADS + 4];     // chunk c of the tile at [c + 4]; halo at [0..3]
  __shared__ unsigned s_ms[SC_MS_WORDS + 1];                                   // module-start bits, strip wbase + i at bit i
  __shared__ int st_module[SC_TILE], st_first[SC_TILE], st_last[SC_TILE];     // staged cluster records, in strip order
  __shared__ unsigned st_charge[SC_TILE];
  __shared__ float st_bary[SC_TILE];
  __shared__ int s_tile, s_mlo, s_mhi, s_kept, s_prefix, s_wsum[SC_THREADS / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  if (tid == 0) { s_tile = (int)atomicAdd(a.ticket, 1u); s_kept = 0; }
  if (tid <= SC_MS_WORDS) s_ms[tid] = 0;
  __syncthreads();
  const int tile = s_tile;
  const int t0 = tile * SC_TILE, t1 = min(t0 + SC_TILE, a.n_strips);
  const int wbase = t0 - SC_HALO;                                             // may be negative for tile 0
  // modules that touch [max(wbase, 0), t1): m in [mlo, mhi)
  if (tid == 0) s_mlo = module_of(a.moff, 0, a.n_modules, max(wbase, 0));
  if (tid == 32) {                                                            // first m in [0, n_modules] with moff[m] >= t1
    int lo = 0, hi = a.n_modules;                                             // moff[0] = 0 < t1 <= moff[n_modules]
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(a.moff + mid) < t1) lo = mid; else hi = mid; }
    s_mhi = hi;
  }
  // threshold bits: own chunk and (threads 0..3) the halo chunks
  const int g0 = t0 + tid * SC_PER;
  unsigned pass, bad;
  strip_bits(a, g0, pass, bad);
  s_pass[tid + 4] = (unsigned char)pass; s_bad[tid + 4] = (unsigned char)bad;
  if (tid < 4) {
    unsigned hp = 0, hb = 0;
    if (tile > 0) strip_bits(a, wbase + tid * SC_PER, hp, hb);
    s_pass[tid] = (unsigned char)hp; s_bad[tid] = (unsigned char)hb;
  }
  __syncthreads();
  const int mlo = s_mlo, mhi = s_mhi;
  for (int m = mlo + tid; m < mhi; m += SC_THREADS) {
    const int pos = __ldg(a.moff + m) - wbase;
    if (pos >= 0 && pos < SC_TILE + SC_HALO) atomicOr(&s_ms[pos >> 5], 1u << (pos & 31));
  }
  __syncthreads();

  // ---- which of my passing strips start a cluster: window bit 32 + k = my strip k, bit 31 = the strip before ...
  unsigned starts = 0;
  if (pass) {
    const unsigned long long wp = (unsigned long long)s_pass[tid] | ((unsigned long long)s_pass[tid + 1] << 8) |
        ((unsigned long long)s_pass[tid + 2] << 16) | ((unsigned long long)s_pass[tid + 3] << 24) | ((unsigned long long)pass << 32);
    const unsigned long long wb = (unsigned long long)s_bad[tid] | ((unsigned long long)s_bad[tid + 1] << 8) |
        ((unsigned long long)s_bad[tid + 2] << 16) | ((unsigned long long)s_bad[tid + 3] << 24) | ((unsigned long long)bad << 32);
    const int wi = tid >> 2, sh = (tid & 3) * 8;
    const unsigned long long wm = ((unsigned long long)s_ms[wi] | ((unsigned long long)s_ms[wi + 1] << 32)) >> sh;
    for (unsigned rest = pass; rest; rest &= rest - 1) {
      const int k = __ffs(rest) - 1;
      int pos = 32 + k, holes = 0, nbad = 0;
      bool is_start = true;
      while (!((wm >> pos) & 1ull) && pos > 0) {          // stop at the first strip of the module
        pos--;
        if ((wp >> pos) & 1ull) { is_start = false; break; }
        if ((wb >> pos) & 1ull) nbad++; else holes++;
        if (holes > a.max_holes || nbad > a.max_bad) break;
      }
      starts |= (unsigned)is_start << k;
    }
  }
  // exclusive scan of the number of starts per thread -> staging slot
  const int ns = __popc(starts);
  int incl = ns;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += v; }
  if (lane == 31) s_wsum[warp] = incl;
  __syncthreads();
  int slot = incl - ns, nstart = 0;
#pragma unroll
  for (int w = 0; w < SC_THREADS / 32; w++) { const int v = s_wsum[w]; if (w < warp) slot += v; nstart += v; }

  // ---- walk each cluster that starts in my chunk, in strip order (R8), and stage its record
  int nkept = 0;
  {
    int m = -1, b = 0, e = 0;
    const double cut = __dmul_rn((double)a.clus_thr, (double)a.clus_thr);
    for (unsigned rest = starts; rest; rest &= rest - 1, slot++) {
      const int g = g0 + __ffs(rest) - 1;
      if (g >= e) { m = module_of(a.moff, mlo, mhi, g); b = __ldg(a.moff + m); e = __ldg(a.moff + m + 1); }
      int j = g, last = g, holes = 0, nbad = 0;
      bool seed = false;
      unsigned long long q2 = 0, s1 = 0; unsigned charge = 0; double n2 = 0.0;
      while (j < e) {
        const unsigned adc = __ldg(a.adc + j); const float nz = __ldg(a.noise + j); const bool bd = __ldg(a.bad + j) != 0;
        if (!bd && (float)adc > a.chan_thr * nz) {
          last = j; holes = 0; nbad = 0;
          seed |= (float)adc > a.seed_thr * nz;
          q2 += adc * adc; charge += adc; s1 += (unsigned long long)adc * (unsigned)(j - b);
          n2 = __dadd_rn(n2, __dmul_rn((double)nz, (double)nz));
        } else {
          if (bd) nbad++; else holes++;
          if (holes > a.max_holes || nbad > a.max_bad) break;
        }
        j++;
      }
      const bool kept = seed && (double)q2 > __dmul_rn(cut, n2) && (long long)charge >= (long long)a.min_charge;
      st_module[slot] = kept ? m : -1;
      if (kept) {
        st_first[slot] = g - b; st_last[slot] = last - b; st_charge[slot] = charge;
        st_bary[slot] = (float)__ddiv_rn(__dmul_rn((double)(2ull * s1 + charge), 0.5), (double)charge);
        nkept++;
      }
    }
  }
  if (nkept) atomicAdd(&s_kept, nkept);
  __syncthreads();

  // ---- decoupled look-back over the tiles: exclusive prefix of the kept counts
  if (tid == 0) {
    const unsigned long long mine = (unsigned)s_kept;
    volatile unsigned long long* st = a.tile_state;
    unsigned excl = 0;
    if (tile > 0) {
      st[tile] = (1ull << 32) | mine;
      for (int i = tile - 1; i >= 0; i--) {
        unsigned long long v;
        do { v = st[i]; } while ((v >> 32) == 0);
        excl += (unsigned)v;
        if ((v >> 32) == 2) break;
      }
    }
    st[tile] = (2ull << 32) | (unsigned long long)(excl + (unsigned)mine);
    s_prefix = (int)excl;
    if (tile == a.n_tiles - 1) *a.n_clusters = (int)(excl + (unsigned)mine);
  }
  __syncthreads();

  // ---- ordered compaction of the staged records
  int base = s_prefix;
  for (int c0 = 0; c0 < nstart; c0 += SC_THREADS) {
    const int s = c0 + tid;
    const bool f = s < nstart && st_module[s] >= 0;
    const unsigned bal = __ballot_sync(0xffffffffu, f);
    __syncthreads();                                     // s_wsum of the previous round has been read
    if (lane == 0) s_wsum[warp] = __popc(bal);
    __syncthreads();
    int off = base + __popc(bal & ((1u << lane) - 1u)), tot = 0;
#pragma unroll
    for (int w = 0; w < SC_THREADS / 32; w++) { const int v = s_wsum[w]; if (w < warp) off += v; tot += v; }
    if (f && off < a.cap) {
      a.o_module[off] = st_module[s]; a.o_first[off] = st_first[s]; a.o_last[off] = st_last[s];
      a.o_charge[off] = st_charge[s]; a.o_bary[off] = st_bary[s];
    }
    base += tot;
  }
}

size_t strips_ws_bytes(int n_strips) {
  const size_t n_tiles = ((size_t)n_strips + SC_TILE - 1) / SC_TILE;
  return align256(n_tiles * sizeof(unsigned long long)) + 256;
}
}  // namespace mkf
using namespace mkf;

extern "C" int mkf_cluster_strips(mkf_ctx* c, const mkf_strips* s, const mkf_strip_params* p, const mkf_clusters* out,
                                  void* ws, size_t ws_bytes, void* stream) {
  if (!c) return MKF_INVALID_ARG;
  if (!s || !p || !out || s->n_strips < 0 || s->n_modules < 0 || out->capacity < 0 || !out->n_clusters)
    return fail(c, MKF_INVALID_ARG, "mkf_cluster_strips: bad argument");
  if (s->n_strips > 2147483647 - 2 * SC_TILE) return fail(c, MKF_UNSUPPORTED, "mkf_cluster_strips: too many strips for one call");
  if (p->max_holes < 0 || p->max_bad < 0 || p->max_holes + p->max_bad > SC_HALO - 1)
    return fail(c, MKF_UNSUPPORTED, "mkf_cluster_strips: max_holes + max_bad must lie in 0..31");
  cudaStream_t st = (cudaStream_t)stream;
  if (s->n_strips == 0 || s->n_modules == 0) {
    cudaError_t e = cudaMemsetAsync(out->n_clusters, 0, sizeof(int), st);
    return e == cudaSuccess ? MKF_OK : cuda_fail(c, e, "mkf_cluster_strips: memset");
  }
  if (!s->module_off || !s->adc || !s->noise || !s->bad ||
      (out->capacity > 0 && (!out->module || !out->first || !out->last || !out->charge || !out->bary)))
    return fail(c, MKF_INVALID_ARG, "mkf_cluster_strips: null pointer");
  if (((uintptr_t)s->adc & 15) || ((uintptr_t)s->noise & 15) || ((uintptr_t)s->bad & 7))
    return fail(c, MKF_INVALID_ARG, "mkf_cluster_strips: adc / noise must be 16-byte aligned, bad 8-byte aligned");
  const size_t need = strips_ws_bytes(s->n_strips);
  if (!ws || ws_bytes < need) return fail(c, MKF_WORKSPACE_TOO_SMALL, "mkf_cluster_strips: workspace too small");
  ScArgs a;
  a.n_modules = s->n_modules; a.n_strips = s->n_strips; a.n_tiles = (s->n_strips + SC_TILE - 1) / SC_TILE;
  a.moff = s->module_off; a.adc = s->adc; a.noise = s->noise; a.bad = s->bad;
  a.seed_thr = p->seed_thr; a.chan_thr = p->chan_thr; a.clus_thr = p->clus_thr;
  a.min_charge = p->min_charge; a.max_holes = p->max_holes; a.max_bad = p->max_bad;
  a.cap = out->capacity; a.o_module = out->module; a.o_first = out->first; a.o_last = out->last;
  a.o_charge = out->charge; a.o_bary = out->bary; a.n_clusters = out->n_clusters;
  a.tile_state = (unsigned long long*)ws;
  a.ticket = (unsigned*)((char*)ws + align256((size_t)a.n_tiles * sizeof(unsigned long long)));
  cudaError_t e = cudaMemsetAsync(ws, 0, need, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "mkf_cluster_strips: memset");
  sc_cluster_kernel<<<a.n_tiles, SC_THREADS, 0, st>>>(a);
  MKF_LAUNCHED(c, "sc_cluster_kernel");
  return MKF_OK;
}
