// mkf_strips.cu — strip clustering (reading R8 of DESIGN.md) in ONE pass over the strips.
//
// HBM-bound: 7 bytes per strip in (adc u16, noise f32, bad u8), 20 bytes per kept cluster out. One CTA takes a tile
// of SC_TILE consecutive strips of the concatenated batch, each thread SC_SUB chunks of 8 consecutive strips with
// 16-byte loads. Tiles do not wait for one another:
//   1. threshold bits (pass / bad) of the tile and of a 32-strip halo to its left, module-start bits from module_off;
//   2. a passing strip starts a cluster iff no passing strip of its module lies within the allowed gap to its left
//      (bit tests on a 40-strip window per chunk);
//   3. the starts are listed in shared memory and walked one per thread, in strip order (the sums of R8 are
//      order-dependent in fp64);
//   4. the kept records of the tile go to staging arrays at a position taken from one global counter;
//   5. sc_scan_tiles_kernel + sc_gather_kernel put the tiles' records in order: (module, first strip).
// (A single-kernel version with a decoupled look-back over the tiles was 2x slower: the tiles of a wave then finish
// together, and loads and arithmetic stop overlapping across CTAs.)
// Nothing here is shared with oracle/.
#include "mkf_ctx.h"
#include <cstdint>

namespace mkf {

#ifndef SC_SUB
#define SC_SUB 4
#endif
constexpr int SC_THREADS = 256, SC_PER = 8, SC_CHUNKS = SC_THREADS * SC_SUB, SC_TILE = SC_CHUNKS * SC_PER, SC_HALO = 32;
constexpr int SC_MS_WORDS = (SC_TILE + SC_HALO) / 32;
#ifndef SC_MIN_BLOCKS
#define SC_MIN_BLOCKS 6
#endif

struct ScArgs {
  int n_modules, n_strips, n_tiles;
  const int* moff; const unsigned short* adc; const float* noise; const unsigned char* bad;
  float seed_thr, chan_thr, clus_thr; int min_charge, max_holes, max_bad;
  int cap; int *o_module, *o_first, *o_last; unsigned* o_charge; float* o_bary; int* n_clusters;
  unsigned* total;                      // clusters found so far = next free record of the staging arrays
  int *tile_cnt, *tile_base;            // [n_tiles]: kept clusters of the tile, where its records are staged
  int stage_cap; int *g_module, *g_first, *g_last; unsigned* g_charge; float* g_bary;     // staging, tile by tile in arrival order
  const int* tile_mod;                  // [n_tiles]: module of the first strip of the tile's window
};

// largest m in [lo, hi) with moff[m] <= g (moff ascending; hi > lo and moff[lo] <= g)
__device__ __forceinline__ int module_of(const int* __restrict__ moff, int lo, int hi, int g) {
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(moff + mid) <= g) lo = mid; else hi = mid;
  }
  return lo;
}

// bit i = byte i of w is non-zero
__device__ __forceinline__ unsigned nonzero_bytes(unsigned w) {
  const unsigned t = (((w & 0x7f7f7f7fu) + 0x7f7f7f7fu) | w) & 0x80808080u;
  return (t * 0x00204081u) >> 28;
}

// (float)adc > t for a 16-bit adc, without the integer-to-float conversion: adc_magic = adc | 0x4b000000 is the bit
// pattern of 2^23 + adc, and 2^23 + t rounded towards zero that of 2^23 + floor(t) for 0 <= t < 2^23, so the signed
// comparison of the patterns is adc > floor(t), which for an integer adc is adc > t. t < 0 gives a smaller (or negative)
// pattern: true; t >= 2^23, inf and NaN give a larger one: false. Exactly the float comparison in every case.
__device__ __forceinline__ bool above_threshold(unsigned adc_magic, float t) {
  return (int)adc_magic > __float_as_int(__fadd_rz(t, 8388608.0f));
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
    bad = nonzero_bytes(bv.x) | (nonzero_bytes(bv.y) << 4);
    unsigned above = 0;
#pragma unroll
    for (int k = 0; k < 8; k++) {
      above |= (unsigned)above_threshold(__byte_perm(aw[k >> 1], 0x4b000000u, (k & 1) ? 0x7632 : 0x7610), a.chan_thr * nz[k]) << k;
    }
    pass = above & ~bad;
  } else {
    for (int k = 0; k < 8 && g0 + k < a.n_strips; k++) {
      const unsigned b = a.bad[g0 + k] != 0;
      bad |= b << k;
      pass |= (unsigned)(!b && (float)a.adc[g0 + k] > a.chan_thr * a.noise[g0 + k]) << k;
    }
  }
}

// tile t -> the module that holds the first strip of its window, max(t * tile_strips - SC_HALO, 0). One thread per module.
__global__ void sc_tile_module_kernel(int n_modules, int n_tiles, int tile_strips, const int* __restrict__ moff, int* __restrict__ tile_mod) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n_modules) return;
  const int b = moff[m], e = moff[m + 1];
  if (e <= b) return;
  if (b == 0) tile_mod[0] = m;
  const int tlo = max((b + SC_HALO + tile_strips - 1) / tile_strips, 1), thi = min((e - 1 + SC_HALO) / tile_strips, n_tiles - 1);
  for (int t = tlo; t <= thi; t++) tile_mod[t] = m;
}

struct ScRecord { int module, first, last; unsigned charge; float bary; };

// largest k in [0, n) with s_off[k] <= g (shared copy of module_off[mlo ..]; s_off[0] <= g)
__device__ __forceinline__ int module_of_shared(const int* s_off, int n, int g) {
  int lo = 0, hi = n;
  while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (s_off[mid] <= g) lo = mid; else hi = mid; }
  return lo;
}

struct ScSums { int last, holes, nbad; bool seed, open; unsigned long long q2, s1; unsigned charge; double n2; };

// one strip of the walk of R8 (strip order); open = false once the gap rule has closed the cluster
__device__ __forceinline__ void sc_strip(const ScArgs& a, ScSums& w, int j, int b, unsigned adc, float nz, bool bd) {
  if (!bd && (float)adc > a.chan_thr * nz) {
    w.last = j; w.holes = 0; w.nbad = 0;
    w.seed |= (float)adc > a.seed_thr * nz;
    w.q2 += adc * adc; w.charge += adc; w.s1 += (unsigned long long)adc * (unsigned)(j - b);
    w.n2 = __dadd_rn(w.n2, __dmul_rn((double)nz, (double)nz));
  } else {
    if (bd) w.nbad++; else w.holes++;
    if (w.holes > a.max_holes || w.nbad > a.max_bad) w.open = false;
  }
}

// R8 in strip order for the cluster that starts at strip g (a passing strip) of module m = [b, e). Returns whether
// it is kept. The first SC_PRE strips are loaded together (one round trip for the usual short cluster).
constexpr int SC_PRE = 4;
__device__ __forceinline__ bool sc_walk(const ScArgs& a, int m, int b, int e, int g, double cut, ScRecord& r) {
  unsigned av[SC_PRE]; float nv[SC_PRE]; unsigned char bv[SC_PRE];
#pragma unroll
  for (int q = 0; q < SC_PRE; q++) {
    const bool in = g + q < e;
    av[q] = in ? __ldg(a.adc + g + q) : 0u; nv[q] = in ? __ldg(a.noise + g + q) : 0.0f; bv[q] = in ? __ldg(a.bad + g + q) : (unsigned char)0;
  }
  ScSums w; w.last = g; w.holes = 0; w.nbad = 0; w.seed = false; w.open = true; w.q2 = 0; w.s1 = 0; w.charge = 0; w.n2 = 0.0;
#pragma unroll
  for (int q = 0; q < SC_PRE; q++)
    if (w.open && g + q < e) sc_strip(a, w, g + q, b, av[q], nv[q], bv[q] != 0);
  for (int j = g + SC_PRE; w.open && j < e; j++) sc_strip(a, w, j, b, __ldg(a.adc + j), __ldg(a.noise + j), __ldg(a.bad + j) != 0);
  if (!(w.seed && (double)w.q2 > __dmul_rn(cut, w.n2) && (long long)w.charge >= (long long)a.min_charge)) return false;
  r.module = m; r.first = g - b; r.last = w.last - b; r.charge = w.charge;
  r.bary = (float)__ddiv_rn(__dmul_rn((double)(2ull * w.s1 + w.charge), 0.5), (double)w.charge);
  return true;
}

// sum and exclusive prefix (for this warp) of the SC_THREADS / 32 per-warp counts in s_w
__device__ __forceinline__ void warp_counts(const int* s_w, int lane, int warp, int& before, int& total) {
  const int v = lane < SC_THREADS / 32 ? s_w[lane] : 0;
  int incl = v;
#pragma unroll
  for (int d = 1; d < SC_THREADS / 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += t; }
  total = __shfl_sync(0xffffffffu, incl, SC_THREADS / 32 - 1);
  before = __shfl_sync(0xffffffffu, incl - v, warp);
}

constexpr int SC_MOFF = SC_THREADS;                       // module offsets of the tile kept in shared memory

__global__ void __launch_bounds__(SC_THREADS, SC_MIN_BLOCKS) sc_cluster_kernel(const ScArgs a) {
  __shared__ unsigned char s_pass[SC_CHUNKS + 4], s_bad[SC_CHUNKS + 4];       // chunk c of the tile at [c + 4]; halo at [0..3]
  __shared__ unsigned s_ms[SC_MS_WORDS + 2];                                   // module-start bits, strip wbase + i at bit i
  __shared__ unsigned short s_start[SC_TILE];                                  // cluster starts of the tile (tile-relative), ascending
  __shared__ int s_moff[SC_MOFF];                                              // module_off[mlo + i]
  __shared__ unsigned long long s_wa[SC_THREADS / 32];
  __shared__ int s_prefix, s_wb[SC_THREADS / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  for (int i = tid; i < SC_MS_WORDS + 2; i += SC_THREADS) s_ms[i] = 0;
  __syncthreads();
  const int tile = blockIdx.x;
  const int t0 = tile * SC_TILE, t1 = min(t0 + SC_TILE, a.n_strips);
  const int wbase = t0 - SC_HALO;                                             // negative for tile 0
  const int mlo = __ldg(a.tile_mod + tile);
  // threshold bits: own chunks (chunk c = sub * SC_THREADS + tid holds strips t0 + 8 c ..) and (threads 0..3) the halo
  unsigned pass[SC_SUB], bad[SC_SUB];
#pragma unroll
  for (int u = 0; u < SC_SUB; u++) {
    const int c = u * SC_THREADS + tid;
    strip_bits(a, t0 + c * SC_PER, pass[u], bad[u]);
    s_pass[c + 4] = (unsigned char)pass[u]; s_bad[c + 4] = (unsigned char)bad[u];
  }
  if (tid < 4) {
    unsigned hp = 0, hb = 0;
    if (tile > 0) strip_bits(a, wbase + tid * SC_PER, hp, hb);
    s_pass[tid] = (unsigned char)hp; s_bad[tid] = (unsigned char)hb;
  }
  // modules that start before the end of the tile: m in [mlo, mhi); their first strips are marked in s_ms
  int mhi = mlo;
  for (int m0 = mlo;; m0 += SC_THREADS) {
    const int m = m0 + tid;
    const int off = m <= a.n_modules ? __ldg(a.moff + m) : 0x7fffffff;
    if (m0 == mlo) s_moff[tid] = off;
    const bool in = m < a.n_modules && off < t1;
    if (in && off >= wbase) atomicOr(&s_ms[(off - wbase) >> 5], 1u << ((off - wbase) & 31));
    const int c = __syncthreads_count(in);
    mhi += c;
    if (c < SC_THREADS) break;
  }
  const bool moff_shared = mhi - mlo < SC_MOFF;        // then s_moff holds module_off[mlo .. mhi]

  // ---- which of my passing strips start a cluster: window bit 32 + k = strip k of the chunk, bit 31 = the strip before ...
  unsigned starts = 0;                                 // 8 bits per chunk
  const bool short_gap = a.max_holes == 0 && a.max_bad <= 1;     // the gap reaches at most two strips back
#pragma unroll
  for (int u = 0; u < SC_SUB; u++) {
    if (pass[u] == 0) continue;
    const int c = u * SC_THREADS + tid;
    if (short_gap) {
      // 16-bit windows: bit 8 + k = strip k of the chunk, bits 0..7 = the chunk before. A passing strip i is linked
      // to the left iff no module starts at i and (i-1 passes, or i-1 is bad, no module starts there and i-2 passes)
      const unsigned wp = (unsigned)s_pass[c + 3] | (pass[u] << 8), wb = (unsigned)s_bad[c + 3] | (bad[u] << 8);
      const int bit = SC_HALO - 8 + 8 * c;
      const unsigned wm = __funnelshift_r(s_ms[bit >> 5], s_ms[(bit >> 5) + 1], bit & 31);
      const unsigned over_bad = a.max_bad ? (wb << 1) & ~(wm << 1) & (wp << 2) : 0u;
      const unsigned linked = ~wm & ((wp << 1) | over_bad);
      starts |= (pass[u] & ~(linked >> 8) & 0xffu) << (8 * u);
      continue;
    }
    const unsigned long long wp = (unsigned long long)s_pass[c] | ((unsigned long long)s_pass[c + 1] << 8) |
        ((unsigned long long)s_pass[c + 2] << 16) | ((unsigned long long)s_pass[c + 3] << 24) | ((unsigned long long)pass[u] << 32);
    const unsigned long long wb = (unsigned long long)s_bad[c] | ((unsigned long long)s_bad[c + 1] << 8) |
        ((unsigned long long)s_bad[c + 2] << 16) | ((unsigned long long)s_bad[c + 3] << 24) | ((unsigned long long)bad[u] << 32);
    const int wi = c >> 2, sh = (c & 3) * 8;
    const unsigned long long wm = ((unsigned long long)s_ms[wi] | ((unsigned long long)s_ms[wi + 1] << 32)) >> sh;
    for (unsigned rest = pass[u]; rest; rest &= rest - 1) {
      const int k = __ffs(rest) - 1, P = 32 + k;
      const unsigned long long below = wp & ((1ull << P) - 1ull);
      bool is_start = true;
      if (below) {                                      // p: the nearest passing strip before P
        const int p = 63 - __clzll((long long)below);
        const unsigned long long upto_p = (2ull << p) - 1ull;
        const int nb = __popcll(wb & ((1ull << P) - 1ull) & ~upto_p);
        const bool boundary = (wm & ((2ull << P) - 1ull) & ~upto_p) != 0;      // a module starts in (p, P]
        is_start = boundary || nb > a.max_bad || (P - p - 1 - nb) > a.max_holes;
      }
      starts |= (unsigned)is_start << (8 * u + k);
    }
  }
  // exclusive scan of the starts per (sub-tile, thread), all sub-tiles at once: 16 bits of a 64-bit word each
  unsigned long long cnt = 0;
#pragma unroll
  for (int u = 0; u < SC_SUB; u++) cnt |= (unsigned long long)__popc((starts >> (8 * u)) & 0xffu) << (16 * u);
  unsigned long long incl = cnt;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const unsigned long long v = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += v; }
  if (lane == 31) s_wa[warp] = incl;
  __syncthreads();
  int nstart;
  {
    const unsigned long long v = lane < SC_THREADS / 32 ? s_wa[lane] : 0ull;
    unsigned long long wi = v;
#pragma unroll
    for (int d = 1; d < SC_THREADS / 32; d <<= 1) { const unsigned long long t = __shfl_up_sync(0xffffffffu, wi, d); if (lane >= d) wi += t; }
    const unsigned long long total = __shfl_sync(0xffffffffu, wi, SC_THREADS / 32 - 1);
    const unsigned long long mine = __shfl_sync(0xffffffffu, wi - v, warp) + incl - cnt;   // starts before me, per sub-tile
    int base = 0;
#pragma unroll
    for (int u = 0; u < SC_SUB; u++) {
      int slot = base + (int)((mine >> (16 * u)) & 0xffffu);
      const int c = u * SC_THREADS + tid;
      for (unsigned rest = (starts >> (8 * u)) & 0xffu; rest; rest &= rest - 1) s_start[slot++] = (unsigned short)(c * SC_PER + __ffs(rest) - 1);
      base += (int)((total >> (16 * u)) & 0xffffu);
    }
    nstart = base;
  }
  __syncthreads();

  // ---- one cluster per thread: walk it; count the kept ones
  const double cut = __dmul_rn((double)a.clus_thr, (double)a.clus_thr);
  const int rounds = (nstart + SC_THREADS - 1) / SC_THREADS;
  auto walk_slot = [&](int s, ScRecord& rec) -> bool {
    if (s >= nstart) return false;
    const int g = t0 + s_start[s];
    int m, b, e;
    if (moff_shared) { const int k = module_of_shared(s_moff, mhi - mlo, g); m = mlo + k; b = s_moff[k]; e = s_moff[k + 1]; }
    else { m = module_of(a.moff, mlo, mhi, g); b = __ldg(a.moff + m); e = __ldg(a.moff + m + 1); }
    return sc_walk(a, m, b, e, g, cut, rec);
  };
  ScRecord rec;
  bool kept = false;
  int kept_before = 0, nkept = 0;                      // (single round) kept clusters of the lower warps; of the tile
  for (int r = 0; r < rounds; r++) {
    kept = walk_slot(r * SC_THREADS + tid, rec);
    const unsigned bal = __ballot_sync(0xffffffffu, kept);
    if (r > 0) __syncthreads();
    if (lane == 0) s_wb[warp] = __popc(bal);
    __syncthreads();
    int tot;
    warp_counts(s_wb, lane, warp, kept_before, tot);
    kept_before += __popc(bal & ((1u << lane) - 1u));
    nkept += tot;
  }

  // ---- room for the tile's records in the staging arrays (tiles arrive in any order; sc_gather_kernel orders them)
  if (tid == 0) {
    const int base = nkept ? (int)atomicAdd(a.total, (unsigned)nkept) : 0;
    s_prefix = base; a.tile_cnt[tile] = nkept; a.tile_base[tile] = base;
  }
  __syncthreads();
  int base = s_prefix;
  if (rounds <= 1) {
    const int off = base + kept_before;
    if (kept && off < a.stage_cap) {
      a.g_module[off] = rec.module; a.g_first[off] = rec.first; a.g_last[off] = rec.last; a.g_charge[off] = rec.charge; a.g_bary[off] = rec.bary;
    }
  } else {                                             // rare: more starts than threads -> walk again, round by round
    for (int r = 0; r < rounds; r++) {
      kept = walk_slot(r * SC_THREADS + tid, rec);
      const unsigned bal = __ballot_sync(0xffffffffu, kept);
      __syncthreads();
      if (lane == 0) s_wb[warp] = __popc(bal);
      __syncthreads();
      int tot;
      warp_counts(s_wb, lane, warp, kept_before, tot);
      const int off = base + kept_before + __popc(bal & ((1u << lane) - 1u));
      if (kept && off < a.stage_cap) {
        a.g_module[off] = rec.module; a.g_first[off] = rec.first; a.g_last[off] = rec.last; a.g_charge[off] = rec.charge; a.g_bary[off] = rec.bary;
      }
      base += tot;
    }
  }
}

// exclusive scan of the kept counts over the tiles (one CTA, one contiguous segment of tiles per thread; n_tiles is
// small: one tile = SC_TILE strips)
constexpr int SC_SCAN_THREADS = 1024;
__global__ void __launch_bounds__(SC_SCAN_THREADS) sc_scan_tiles_kernel(int n_tiles, const int* __restrict__ tile_cnt,
                                                                        int* __restrict__ tile_out, int* __restrict__ n_clusters) {
  __shared__ int s_w[SC_SCAN_THREADS / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int seg = (n_tiles + SC_SCAN_THREADS - 1) / SC_SCAN_THREADS;
  const int i0 = min(tid * seg, n_tiles), i1 = min(i0 + seg, n_tiles);
  int sum = 0;
  for (int i = i0; i < i1; i++) sum += tile_cnt[i];
  int incl = sum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += t; }
  if (lane == 31) s_w[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    const int w = s_w[lane];
    int wi = w;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, wi, d); if (lane >= d) wi += t; }
    s_w[lane] = wi - w;
    if (lane == 31) *n_clusters = wi;
  }
  __syncthreads();
  int run = s_w[warp] + incl - sum;
  for (int i = i0; i < i1; i++) { tile_out[i] = run; run += tile_cnt[i]; }
}

// staged records -> output arrays in tile order = (module, first strip) order. One warp per tile.
__global__ void __launch_bounds__(256) sc_gather_kernel(const ScArgs a, const int* __restrict__ tile_out) {
  const int tile = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (tile >= a.n_tiles) return;
  const int n = a.tile_cnt[tile], src = a.tile_base[tile], dst = tile_out[tile];
  for (int i = lane; i < n; i += 32) {
    if (src + i < a.stage_cap && dst + i < a.cap) {
      a.o_module[dst + i] = a.g_module[src + i]; a.o_first[dst + i] = a.g_first[src + i]; a.o_last[dst + i] = a.g_last[src + i];
      a.o_charge[dst + i] = a.g_charge[src + i]; a.o_bary[dst + i] = a.g_bary[src + i];
    }
  }
}

// workspace: total counter | tile_mod, tile_cnt, tile_base, tile_out [n_tiles] | staging 5 x capacity
size_t strips_ws_bytes(int n_strips, int capacity) {
  const size_t n_tiles = ((size_t)n_strips + SC_TILE - 1) / SC_TILE;
  return 256 + 4 * align256(n_tiles * sizeof(int)) + 5 * align256((size_t)capacity * sizeof(int));
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
  const size_t need = strips_ws_bytes(s->n_strips, out->capacity);
  if (!ws || ws_bytes < need) return fail(c, MKF_WORKSPACE_TOO_SMALL, "mkf_cluster_strips: workspace too small");
  if ((uintptr_t)ws & 15) return fail(c, MKF_INVALID_ARG, "mkf_cluster_strips: workspace must be 16-byte aligned");
  ScArgs a;
  a.n_modules = s->n_modules; a.n_strips = s->n_strips; a.n_tiles = (s->n_strips + SC_TILE - 1) / SC_TILE;
  a.moff = s->module_off; a.adc = s->adc; a.noise = s->noise; a.bad = s->bad;
  a.seed_thr = p->seed_thr; a.chan_thr = p->chan_thr; a.clus_thr = p->clus_thr;
  a.min_charge = p->min_charge; a.max_holes = p->max_holes; a.max_bad = p->max_bad;
  a.cap = out->capacity; a.o_module = out->module; a.o_first = out->first; a.o_last = out->last;
  a.o_charge = out->charge; a.o_bary = out->bary; a.n_clusters = out->n_clusters;
  char* w = (char*)ws;
  const size_t tb = align256((size_t)a.n_tiles * sizeof(int)), cb = align256((size_t)out->capacity * sizeof(int));
  a.total = (unsigned*)w; w += 256;
  int* tile_mod = (int*)w; w += tb; a.tile_mod = tile_mod;
  a.tile_cnt = (int*)w; w += tb; a.tile_base = (int*)w; w += tb;
  int* tile_out = (int*)w; w += tb;
  a.stage_cap = out->capacity;
  a.g_module = (int*)w; w += cb; a.g_first = (int*)w; w += cb; a.g_last = (int*)w; w += cb;
  a.g_charge = (unsigned*)w; w += cb; a.g_bary = (float*)w;
  cudaError_t e = cudaMemsetAsync(a.total, 0, 256, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "mkf_cluster_strips: memset");
  sc_tile_module_kernel<<<(a.n_modules + 255) / 256, 256, 0, st>>>(a.n_modules, a.n_tiles, SC_TILE, a.moff, tile_mod);
  MKF_LAUNCHED(c, "sc_tile_module_kernel");
  sc_cluster_kernel<<<a.n_tiles, SC_THREADS, 0, st>>>(a);
  MKF_LAUNCHED(c, "sc_cluster_kernel");
  sc_scan_tiles_kernel<<<1, SC_SCAN_THREADS, 0, st>>>(a.n_tiles, a.tile_cnt, tile_out, a.n_clusters);
  MKF_LAUNCHED(c, "sc_scan_tiles_kernel");
  sc_gather_kernel<<<(a.n_tiles + 7) / 8, 256, 0, st>>>(a, tile_out);
  MKF_LAUNCHED(c, "sc_gather_kernel");
  return MKF_OK;
}
