// mkf_hit_index.cu — a1 / C8: per (event, layer) phi/eta-binned hit index ("data preparation").
//
// Counting sort over the global bin space (segment = event*n_layers + layer, bin = ie*n_phi + ip):
//   1. hi_key_count : one CTA per segment; bin key per hit in fp64 (U12), count per bin (global atomics on a
//                     mostly empty table), per-segment max hit variances (block reduction, no atomics);
//   2. hi_scan_*    : exclusive prefix sum of the counts (reduce / scan-of-partials / downsweep);
//   3. hi_place     : scatter hit ids to their bins (atomic cursor);
//   4. hi_sort_bins : each bin's ids sorted ascending -> the order is the unique stable order (C8) whatever
//                     order the atomics ran in;
//   5. hi_pack      : the hits in sorted order, positions (16 B) and covariances (32 B) in two contiguous blocks,
//                     so that a bin scan reads contiguous memory.
// That five-kernel path serves the masked index (R9) and bin grids too large for shared memory. The plain index runs
// as ONE kernel, hi_fused_kernel (one CTA per segment): the hits of a segment occupy the same range of positions before
// and after sorting, so its bin offsets are layer_off + a prefix over the segment's own bins, computed in shared
// memory (10 KB for 63 x 40 bins: the occupancy is bounded by threads, not by shared memory); ids are scattered with
// an atomic cursor into a scratch list, and every hit then takes as its place in the bin the number of smaller ids it
// finds there, writing its id and its packed record; the segment is read from HBM once (the later passes hit L2).
// HBM-bound; algorithmic bytes per hit are listed in DESIGN.md §6.
#include <atomic>
#include "mkf_ctx.h"
#include "mkf_scan.cuh"

using namespace mkf;

namespace {

constexpr int HI_BLOCK = 256;

struct HiArgs {
  HitsDev hits; int n_layers, n_phi, n_eta;
  int* key;            // [n_hits] bin inside the segment
  int* tmp_id;         // [n_hits] ids by bin, any order inside a bin (single-kernel path)
  unsigned* cnt;       // [n_bins_total] counts, later the scatter cursors
  unsigned* bin_off; int* sorted_id; float* vmax; float4* packed;
  const unsigned char* mask;     // R9: hits left out of the index (NULL: none)
  size_t n_bins;
};

__device__ __forceinline__ int phi_bin_d(double phi, int nphi) {
  const double PI = 3.14159265358979323846;
  int ip = (int)floor((phi + PI) * (double)nphi / (2.0 * PI));
  if (ip >= nphi) ip -= nphi;
  if (ip < 0) ip = 0;
  return ip;
}
__device__ __forceinline__ int eta_bin_d(double eta, double lo, double hi, int neta) {
  int ie = (int)floor((eta - lo) * (double)neta / (hi - lo));
  if (ie < 0) ie = 0;
  if (ie > neta - 1) ie = neta - 1;
  return ie;
}

__global__ void __launch_bounds__(HI_BLOCK) hi_key_count(const __grid_constant__ GeomDev g, const __grid_constant__ HiArgs a) {
  const int seg = blockIdx.x;
  const int ev = seg / a.n_layers, l = seg - ev * a.n_layers;
  const int b = a.hits.layer_off[ev * (a.n_layers + 1) + l], e = a.hits.layer_off[ev * (a.n_layers + 1) + l + 1];
  const double elo = (double)g.layers[l].eta_lo, ehi = (double)g.layers[l].eta_hi;
  const size_t nh = (size_t)a.hits.n_hits;
  const size_t bin0 = (size_t)seg * (size_t)(a.n_phi * a.n_eta);
  float vxy = 0.f, vzz = 0.f;
  for (int i = b + threadIdx.x; i < e; i += HI_BLOCK) {
    if (a.mask && a.mask[i]) { a.key[i] = -1; continue; }
    const double x = (double)a.hits.x[i], y = (double)a.hits.y[i], z = (double)a.hits.z[i];
    const int ip = phi_bin_d(atan2(y, x), a.n_phi);
    const int ie = eta_bin_d(asinh(z / sqrt(x * x + y * y)), elo, ehi, a.n_eta);
    const int key = ie * a.n_phi + ip;
    a.key[i] = key;
    atomicAdd(&a.cnt[bin0 + key], 1u);
    // larger eigenvalue of the xy block of V in round-to-nearest fp32 without contraction (bit-exact with C8)
    const float vxx = a.hits.V[i], vxyv = a.hits.V[nh + i], vyy = a.hits.V[2 * nh + i];
    const float hs = __fmul_rn(0.5f, __fadd_rn(vxx, vyy)), hd = __fmul_rn(0.5f, __fsub_rn(vxx, vyy));
    const float ev1 = __fadd_rn(hs, __fsqrt_rn(__fadd_rn(__fmul_rn(hd, hd), __fmul_rn(vxyv, vxyv))));
    vxy = fmaxf(vxy, ev1);
    vzz = fmaxf(vzz, a.hits.V[5 * nh + i]);
  }
  __shared__ float s_xy[HI_BLOCK / 32], s_zz[HI_BLOCK / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    vxy = fmaxf(vxy, __shfl_xor_sync(0xffffffffu, vxy, o));
    vzz = fmaxf(vzz, __shfl_xor_sync(0xffffffffu, vzz, o));
  }
  if ((threadIdx.x & 31) == 0) { s_xy[threadIdx.x >> 5] = vxy; s_zz[threadIdx.x >> 5] = vzz; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < HI_BLOCK / 32; w++) { vxy = fmaxf(vxy, s_xy[w]); vzz = fmaxf(vzz, s_zz[w]); }
    a.vmax[2 * (size_t)seg] = vxy; a.vmax[2 * (size_t)seg + 1] = vzz;
  }
}

__global__ void __launch_bounds__(HI_BLOCK) hi_place(const __grid_constant__ HiArgs a) {
  const int seg = blockIdx.x;
  const int ev = seg / a.n_layers, l = seg - ev * a.n_layers;
  const int b = a.hits.layer_off[ev * (a.n_layers + 1) + l], e = a.hits.layer_off[ev * (a.n_layers + 1) + l + 1];
  const size_t bin0 = (size_t)seg * (size_t)(a.n_phi * a.n_eta);
  for (int i = b + threadIdx.x; i < e; i += HI_BLOCK) {
    const int key = a.key[i];
    if (key < 0) continue;
    const unsigned pos = atomicAdd(&a.cnt[bin0 + key], 1u);
    a.sorted_id[pos] = i;
  }
}

// one thread per bin: ascending ids (insertion sort for the usual handful, heap sort for crowded edge bins)
__global__ void __launch_bounds__(HI_BLOCK) hi_sort_bins(const unsigned* __restrict__ bin_off, size_t n_bins, int* sorted_id) {
  const size_t bin = (size_t)blockIdx.x * HI_BLOCK + threadIdx.x;
  if (bin >= n_bins) return;
  const unsigned b = bin_off[bin], e = bin_off[bin + 1];
  const int len = (int)(e - b);
  if (len < 2) return;
  int* v = sorted_id + b;
  if (len <= 24) {
    for (int i = 1; i < len; i++) {
      const int x = v[i];
      int j = i - 1;
      while (j >= 0 && v[j] > x) { v[j + 1] = v[j]; j--; }
      v[j + 1] = x;
    }
    return;
  }
  auto sift = [&](int start, int end) {
    int root = start;
    while (2 * root + 1 <= end) {
      int child = 2 * root + 1;
      if (child + 1 <= end && v[child] < v[child + 1]) child++;
      if (v[root] < v[child]) { const int t = v[root]; v[root] = v[child]; v[child] = t; root = child; }
      else return;
    }
  };
  for (int s = (len - 2) / 2; s >= 0; s--) sift(s, len - 1);
  for (int end = len - 1; end > 0; end--) { const int t = v[0]; v[0] = v[end]; v[end] = t; sift(0, end - 1); }
}

__global__ void __launch_bounds__(HI_BLOCK) hi_pack(const __grid_constant__ HiArgs a) {
  const int t = blockIdx.x * HI_BLOCK + threadIdx.x;
  if (t >= a.hits.n_hits || (unsigned)t >= a.bin_off[a.n_bins]) return;       // masked hits are not in sorted_id
  const int id = a.sorted_id[t];
  const size_t nh = (size_t)a.hits.n_hits;
  const float* V = a.hits.V;
  // positions first (16 B per hit, what the window scan reads for every hit), covariances behind them (32 B per
  // hit, read only for the hits that survive the position test)
  a.packed[t] = make_float4(a.hits.x[id], a.hits.y[id], a.hits.z[id], __int_as_float(id));
  float4* o = a.packed + packed_cov_off(a.hits.n_hits) + (size_t)2 * t;
  o[0] = make_float4(V[id], V[nh + id], V[2 * nh + id], V[3 * nh + id]);
  o[1] = make_float4(V[4 * nh + id], V[5 * nh + id], a.hits.module ? __int_as_float(a.hits.module[id]) : 0.f, 0.f);
}


// ---- the plain index in one kernel ------------------------------------------------------------------------------------
// threads per segment, CTAs per SM, ids of a segment kept in shared memory between the scatter and the ranking (the rest:
// workspace): for segments of up to / beyond 4096 hits on average
// (measured on configs[2] / [3] / [4]: 256 x 4 CTAs and 1024 x 1: 0.16 / 0.66 / 0.76 ms; 256 x 6 with 6144 ids and 512 x 3:
// 0.18 / 0.76 / 1.13; 256 x 5 with 8192 ids and 512 x 2: 0.17 / 0.70 / 0.94: more segments in flight than L2 holds cost more than
// the occupancy gives)
#define MKF_HF_S 256, 4, 10240
#define MKF_HF_L 1024, 1, 10240
template <int B, int M, int T> struct HfCfg { static constexpr int block = B, minb = M, tmpcap = T; };
using HfSmall = HfCfg<MKF_HF_S>;
using HfLarge = HfCfg<MKF_HF_L>;

// Bin key of a hit, identical to the fp64 evaluation of C8 (U12): fp32 first; the fp64 formulas only when the fp32
// value lies within 1e-3 bin widths of a bin edge (fp32 atan2f / asinhf are good to a few 1e-7 in value, 2e-5 in bin
// units, so outside that margin both evaluations floor to the same bin).
__device__ __forceinline__ int bin_key(float xf, float yf, float zf, float elo_f, float ehi_f, int n_phi, int n_eta) {
  const float PI = 3.14159265358979323846f;
  const float bp = (atan2f(yf, xf) + PI) * ((float)n_phi * (1.f / (2.f * PI)));
  const float be = (asinhf(zf * rsqrtf(fmaf(xf, xf, yf * yf))) - elo_f) * ((float)n_eta / (ehi_f - elo_f));
  int ip, ie;
  if (fabsf(bp - rintf(bp)) > 1e-3f && bp > 0.f && bp < (float)n_phi) ip = (int)bp;
  else ip = phi_bin_d(atan2((double)yf, (double)xf), n_phi);
  if (fabsf(be - rintf(be)) > 1e-3f && be > 0.f && be < (float)n_eta) ie = (int)be;
  else if (be < -1.f) ie = 0;
  else if (be > (float)n_eta + 1.f) ie = n_eta - 1;
  else {
    const double x = (double)xf, y = (double)yf, z = (double)zf;
    ie = eta_bin_d(asinh(z / sqrt(x * x + y * y)), (double)elo_f, (double)ehi_f, n_eta);
  }
  return ie * n_phi + ip;
}

// One CTA per segment, bin counts of the segment in shared memory:
//   A  key per hit (kept in the workspace), count per bin, per-segment max hit variances;
//   -  exclusive prefix over the segment's bins -> bin_off (= layer_off + prefix) and the scatter cursors;
//   B  ids scattered to their bins in a scratch list (atomic cursor: any order inside a bin);
//   C  every hit counts the ids of its bin that are smaller than its own: that rank is its place in the bin (the unique
//      stable order of C8, no sort and no dependent probing: the bin's few ids are independent loads); it writes its id
//      and its packed record there. Hits are read in id order (coalesced) in every pass; two hits per thread and
//      iteration keep more loads in flight.
template <class CFG>
__global__ void __launch_bounds__(CFG::block, CFG::minb) hi_fused_kernel(const __grid_constant__ GeomDev g, const __grid_constant__ HiArgs a) {
  constexpr int HF_BLOCK = CFG::block, HF_WARPS = HF_BLOCK / 32, HF_TMPCAP = CFG::tmpcap;
  extern __shared__ unsigned hf_cnt[];                        // [nb] counts, then cursors; [HF_TMPCAP] ids by bin
  __shared__ float s_xy[HF_WARPS], s_zz[HF_WARPS];
  __shared__ unsigned s_ws[HF_WARPS];
  const int seg = blockIdx.x;
  const int nb = a.n_phi * a.n_eta;
  int* s_tmp = reinterpret_cast<int*>(hf_cnt + nb);
  unsigned short* s_tmp16 = reinterpret_cast<unsigned short*>(s_tmp);     // the same room holds twice as many ids as 16-bit
                                                                          // offsets from the segment's first hit
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int ev = seg / a.n_layers, l = seg - ev * a.n_layers;
  const int b = a.hits.layer_off[ev * (a.n_layers + 1) + l], e = a.hits.layer_off[ev * (a.n_layers + 1) + l + 1];
  const bool ids16 = e - b <= 65536;                          // (uniform in the CTA)
  for (int k = tid; k < nb; k += HF_BLOCK) hf_cnt[k] = 0u;
  __syncthreads();
  const float elo = g.layers[l].eta_lo, ehi = g.layers[l].eta_hi;
  const size_t nh = (size_t)a.hits.n_hits;
  const float* V = a.hits.V;
  float vxy = 0.f, vzz = 0.f;
  for (int i0 = b + tid; i0 < e; i0 += 2 * HF_BLOCK) {
    const int i1 = i0 + HF_BLOCK;
    const bool two = i1 < e;
    const int j1 = two ? i1 : i0;
    const float x0 = a.hits.x[i0], y0 = a.hits.y[i0], z0 = a.hits.z[i0], x1 = a.hits.x[j1], y1 = a.hits.y[j1], z1 = a.hits.z[j1];
    const float p0 = V[i0], q0 = V[nh + i0], r0 = V[2 * nh + i0], t0 = V[5 * nh + i0];
    const float p1 = V[j1], q1 = V[nh + j1], r1 = V[2 * nh + j1], t1 = V[5 * nh + j1];
    const int key0 = bin_key(x0, y0, z0, elo, ehi, a.n_phi, a.n_eta);
    a.key[i0] = key0;
    atomicAdd(&hf_cnt[key0], 1u);
    if (two) {
      const int key1 = bin_key(x1, y1, z1, elo, ehi, a.n_phi, a.n_eta);
      a.key[i1] = key1;
      atomicAdd(&hf_cnt[key1], 1u);
    }
    // larger eigenvalue of the xy block of V in round-to-nearest fp32 without contraction (bit-exact with C8)
    {
      const float hs = __fmul_rn(0.5f, __fadd_rn(p0, r0)), hd = __fmul_rn(0.5f, __fsub_rn(p0, r0));
      vxy = fmaxf(vxy, __fadd_rn(hs, __fsqrt_rn(__fadd_rn(__fmul_rn(hd, hd), __fmul_rn(q0, q0)))));
      vzz = fmaxf(vzz, t0);
    }
    {
      const float hs = __fmul_rn(0.5f, __fadd_rn(p1, r1)), hd = __fmul_rn(0.5f, __fsub_rn(p1, r1));
      vxy = fmaxf(vxy, __fadd_rn(hs, __fsqrt_rn(__fadd_rn(__fmul_rn(hd, hd), __fmul_rn(q1, q1)))));
      vzz = fmaxf(vzz, t1);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    vxy = fmaxf(vxy, __shfl_xor_sync(0xffffffffu, vxy, o));
    vzz = fmaxf(vzz, __shfl_xor_sync(0xffffffffu, vzz, o));
  }
  if (lane == 0) { s_xy[w] = vxy; s_zz[w] = vzz; }
  __syncthreads();
  if (tid == 0) {
    for (int k = 1; k < HF_WARPS; k++) { vxy = fmaxf(vxy, s_xy[k]); vzz = fmaxf(vzz, s_zz[k]); }
    a.vmax[2 * (size_t)seg] = vxy; a.vmax[2 * (size_t)seg + 1] = vzz;
  }
  // exclusive prefix of the counts over the bins (blocked: thread t owns bins [t * pb, (t + 1) * pb))
  {
    const int pb = (nb + HF_BLOCK - 1) / HF_BLOCK;
    const int k0 = min(tid * pb, nb), k1 = min(k0 + pb, nb);
    unsigned sum = 0;
    for (int k = k0; k < k1; k++) sum += hf_cnt[k];
    unsigned inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned t2 = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t2; }
    if (lane == 31) s_ws[w] = inc;
    __syncthreads();
    unsigned base = 0;
    for (int q = 0; q < w; q++) base += s_ws[q];
    unsigned run = (unsigned)b + base + inc - sum;
    unsigned* bo = a.bin_off + (size_t)seg * nb;
    for (int k = k0; k < k1; k++) { const unsigned c = hf_cnt[k]; hf_cnt[k] = run; bo[k] = run; run += c; }
    if (seg == gridDim.x - 1 && tid == 0) a.bin_off[a.n_bins] = (unsigned)a.hits.n_hits;
  }
  __syncthreads();
  for (int i = b + tid; i < e; i += HF_BLOCK) {
    const unsigned pos = atomicAdd(&hf_cnt[a.key[i]], 1u);
    const unsigned o = pos - (unsigned)b;
    if (ids16) { if (o < 2u * HF_TMPCAP) s_tmp16[o] = (unsigned short)(i - b); else a.tmp_id[pos] = i; }
    else { if (o < (unsigned)HF_TMPCAP) s_tmp[o] = i; else a.tmp_id[pos] = i; }
  }
  __syncthreads();                                            // cursor[k] is now the end of bin k
  // rank of id i among the ids of its bin: four independent loads per round (a bin holds a handful of ids)
  auto place = [&](int i, int key) -> unsigned {
    const unsigned kb = key == 0 ? (unsigned)b : hf_cnt[key - 1], ke = hf_cnt[key];
    unsigned rank = 0;
    auto at = [&](unsigned q) -> int {
      const unsigned o = q - (unsigned)b;
      if (ids16) return o < 2u * HF_TMPCAP ? b + (int)s_tmp16[o] : a.tmp_id[q];
      return o < (unsigned)HF_TMPCAP ? s_tmp[o] : a.tmp_id[q];
    };
    for (unsigned q = kb; q < ke; q += 4) {
      const int v0 = at(q);
      const int v1 = q + 1 < ke ? at(q + 1) : 0x7fffffff;
      const int v2 = q + 2 < ke ? at(q + 2) : 0x7fffffff;
      const int v3 = q + 3 < ke ? at(q + 3) : 0x7fffffff;
      rank += (v0 < i ? 1u : 0u) + (v1 < i ? 1u : 0u) + (v2 < i ? 1u : 0u) + (v3 < i ? 1u : 0u);
    }
    return kb + rank;
  };
  auto write = [&](int i, unsigned t, float x, float y, float z, float v0, float v1, float v2, float v3, float v4, float v5) {
    a.sorted_id[t] = i;
    if (a.packed) {
      a.packed[t] = make_float4(x, y, z, __int_as_float(i));
      float4* o = a.packed + packed_cov_off(a.hits.n_hits) + (size_t)2 * t;
      const float md = a.hits.module ? __int_as_float(a.hits.module[i]) : 0.f;
      // one 32-byte store where the block is sector-aligned: a scattered whole-sector write needs no fill from DRAM
      if (((size_t)o & 31) == 0)
        asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" :: "l"(o), "f"(v0), "f"(v1), "f"(v2), "f"(v3), "f"(v4), "f"(v5), "f"(md), "f"(0.f) : "memory");
      else { o[0] = make_float4(v0, v1, v2, v3); o[1] = make_float4(v4, v5, md, 0.f); }
    }
  };
  for (int i0 = b + tid; i0 < e; i0 += 2 * HF_BLOCK) {
    const int i1 = i0 + HF_BLOCK;
    const bool two = i1 < e;
    const int j1 = two ? i1 : i0;
    const int key0 = a.key[i0], key1 = a.key[j1];
    const float x0 = a.hits.x[i0], y0 = a.hits.y[i0], z0 = a.hits.z[i0], x1 = a.hits.x[j1], y1 = a.hits.y[j1], z1 = a.hits.z[j1];
    float u0[6], u1[6];
    if (a.packed) {
#pragma unroll
      for (int k = 0; k < 6; k++) { u0[k] = V[(size_t)k * nh + i0]; u1[k] = V[(size_t)k * nh + j1]; }
    }
    const unsigned t0 = place(i0, key0), t1 = place(j1, key1);
    write(i0, t0, x0, y0, z0, u0[0], u0[1], u0[2], u0[3], u0[4], u0[5]);
    if (two) write(i1, t1, x1, y1, z1, u1[0], u1[1], u1[2], u1[3], u1[4], u1[5]);
  }
}

}  // namespace

namespace mkf {
size_t hit_index_ws_bytes(const mkf_ctx* c, int n_events, int n_hits) {
  const size_t nbins = (size_t)n_events * c->g.n_layers * c->g.n_phi * c->g.n_eta;
  return 2 * align256((size_t)n_hits * 4) + align256(nbins * 4) + scan_partial_bytes(nbins);
}
}  // namespace mkf

extern "C" int mkf_build_hit_index(mkf_ctx* c, const mkf_hits* h, mkf_hit_index* out, void* ws, size_t ws_bytes, void* stream) {
  return mkf_build_hit_index_masked(c, h, nullptr, out, ws, ws_bytes, stream);
}

extern "C" int mkf_build_hit_index_masked(mkf_ctx* c, const mkf_hits* h, const unsigned char* mask, mkf_hit_index* out, void* ws,
                                          size_t ws_bytes, void* stream) {
  if (!c) return MKF_INVALID_ARG;
  if (!h || !out || !out->bin_off || !out->sorted_id || !out->vmax || !h->layer_off)
    return fail(c, MKF_INVALID_ARG, "mkf_build_hit_index: null argument");
  if (h->n_events < 1 || h->n_hits < 0) return fail(c, MKF_INVALID_ARG, "mkf_build_hit_index: bad sizes");
  if (h->n_hits >= (1 << 28)) return fail(c, MKF_UNSUPPORTED, "mkf_build_hit_index: n_hits >= 2^28");
  if (h->n_hits > 0 && (!h->x || !h->y || !h->z || !h->V)) return fail(c, MKF_INVALID_ARG, "mkf_build_hit_index: null hit array");
  const size_t need = hit_index_ws_bytes(c, h->n_events, h->n_hits);
  if (ws_bytes < need || (need && !ws)) return fail(c, MKF_WORKSPACE_TOO_SMALL, "mkf_build_hit_index: workspace too small");
  cudaStream_t st = (cudaStream_t)stream;
  const int nseg = h->n_events * c->g.n_layers;
  const size_t nbins = (size_t)nseg * c->g.n_phi * c->g.n_eta;
  char* w = (char*)ws;
  HiArgs a;
  a.hits = hits_dev(h); a.n_layers = c->g.n_layers; a.n_phi = c->g.n_phi; a.n_eta = c->g.n_eta;
  a.key = (int*)w; w += align256((size_t)h->n_hits * 4);
  a.tmp_id = (int*)w; w += align256((size_t)h->n_hits * 4);
  a.cnt = (unsigned*)w; w += align256(nbins * 4);
  unsigned* partial = (unsigned*)w;
  a.bin_off = out->bin_off; a.sorted_id = out->sorted_id; a.vmax = out->vmax; a.packed = (float4*)out->packed;
  a.mask = mask; a.n_bins = nbins;
  const size_t cnt_smem = (size_t)c->g.n_phi * c->g.n_eta * 4;
  // One kernel while the counts fit in shared memory (measured against the five kernels: 0.16 / 0.34 ms on configs[2],
  // 0.65 / 1.37 on configs[3], 0.77 / 1.64 on configs[4]); 256 threads per segment up to 4096 hits per segment on
  // average, 1024 beyond (configs[4], 7.6 k hits per segment: 2.1 ms with 256 threads).
  const int mode = (size_t)h->n_hits <= (size_t)nseg * 4096 ? 1 : 2;
  if (!mask && cnt_smem <= 64 * 1024) {
    if (h->n_hits == 0) {                                      // nothing to place: all offsets are zero
      cudaError_t e0 = cudaMemsetAsync(a.bin_off, 0, (nbins + 1) * 4, st);
      if (e0 == cudaSuccess) e0 = cudaMemsetAsync(a.vmax, 0, (size_t)nseg * 8, st);
      if (e0 != cudaSuccess) return cuda_fail(c, e0, "mkf_build_hit_index: memset");
      return MKF_OK;
    }
    const size_t smem_s = cnt_smem + (size_t)HfSmall::tmpcap * 4, smem_l = cnt_smem + (size_t)HfLarge::tmpcap * 4;
    {
      cudaError_t e1 = cudaFuncSetAttribute(hi_fused_kernel<HfSmall>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_s);
      if (e1 == cudaSuccess) e1 = cudaFuncSetAttribute(hi_fused_kernel<HfLarge>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_l);
      if (e1 != cudaSuccess) return cuda_fail(c, e1, "mkf_build_hit_index: shared memory attribute");
    }
    if (mode == 2) hi_fused_kernel<HfLarge><<<nseg, HfLarge::block, smem_l, st>>>(c->g, a);
    else hi_fused_kernel<HfSmall><<<nseg, HfSmall::block, smem_s, st>>>(c->g, a);
    MKF_LAUNCHED(c, "hi_fused_kernel");
    return MKF_OK;
  }
  cudaError_t e = cudaMemsetAsync(a.cnt, 0, nbins * 4, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "mkf_build_hit_index: memset");
  hi_key_count<<<nseg, HI_BLOCK, 0, st>>>(c->g, a);
  MKF_LAUNCHED(c, "hi_key_count");
  { const int rc = exclusive_scan_u32(c, a.cnt, nbins, partial, a.bin_off, mask ? SCAN_TOTAL_UNKNOWN : (unsigned)h->n_hits, st); if (rc) return rc; }
  if (h->n_hits > 0) {
    hi_place<<<nseg, HI_BLOCK, 0, st>>>(a);
    MKF_LAUNCHED(c, "hi_place");
    hi_sort_bins<<<(unsigned)((nbins + HI_BLOCK - 1) / HI_BLOCK), HI_BLOCK, 0, st>>>(a.bin_off, nbins, a.sorted_id);
    MKF_LAUNCHED(c, "hi_sort_bins");
    if (a.packed) {
      hi_pack<<<(h->n_hits + HI_BLOCK - 1) / HI_BLOCK, HI_BLOCK, 0, st>>>(a);
      MKF_LAUNCHED(c, "hi_pack");
    }
  }
  return MKF_OK;
}

// ---- R9: the hits of high-quality tracks, masked for the next iteration ------------
namespace {
__global__ void __launch_bounds__(256) mh_mask_kernel(int n, int n_hits, const int* __restrict__ hit_ids, int mpl,
                                                      const int* __restrict__ nhits, const float* __restrict__ chi2,
                                                      const unsigned char* __restrict__ keep, int min_hits, float max_chi2_ndf,
                                                      unsigned char* mask) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (keep && !keep[i]) return;
  const int nh = nhits[i];
  if (nh < min_hits) return;
  if (!(chi2[i] <= __fmul_rn(max_chi2_ndf, (float)(2 * nh - 5)))) return;
  for (int s = 0; s < mpl; s++) {
    const int hid = hit_ids[(size_t)s * n + i];              // coalesced: plane-major
    if (hid >= 0 && hid < n_hits) mask[hid] = 1;             // every writer writes 1
  }
}
}  // namespace

extern "C" int mkf_mask_hits(mkf_ctx* c, int n, int n_hits, const int* hit_ids, int max_plan_len, const int* nhits, const float* chi2,
                             const unsigned char* keep, int min_hits, float max_chi2_ndf, unsigned char* mask, void* stream) {
  if (!c) return MKF_INVALID_ARG;
  if (n < 0 || n_hits < 0 || max_plan_len < 1) return fail(c, MKF_INVALID_ARG, "mkf_mask_hits: bad sizes");
  if (n == 0) return MKF_OK;
  if (!hit_ids || !nhits || !chi2 || (n_hits > 0 && !mask)) return fail(c, MKF_INVALID_ARG, "mkf_mask_hits: null argument");
  mh_mask_kernel<<<(n + 255) / 256, 256, 0, (cudaStream_t)stream>>>(n, n_hits, hit_ids, max_plan_len, nhits, chi2, keep, min_hits,
                                                                    max_chi2_ndf, mask);
  MKF_LAUNCHED(c, "mh_mask_kernel");
  return MKF_OK;
}

// ---- the plain hit index without any caller- or library-allocated scratch ----------------------------------------
// For callers that cannot allocate (CUDA graph capture, tight serving loops): the scratch of hi_fused_kernel (the
// key and the scattered id of every hit, 2 x 4 B per hit) lives in a file-scope device array of
// 2 x MKF_STATIC_MAX_HITS ints = 8 MiB, which every GPU that loads the library holds until exit. All calls on a device
// share it: calls that overlap on the GPU race. Nothing in it has to start at zero (a call reads only words it has
// written itself first), so it is not cleared between calls.
namespace {
static __device__ __align__(256) int g_hi_static_scratch[2 * (size_t)MKF_STATIC_MAX_HITS];

constexpr int HI_MAX_DEVICES = 64;
std::atomic<int*> g_hi_static_ptr[HI_MAX_DEVICES];   // device address of the array per device (host code sees only a stand-in); null: not resolved yet

// The array's device address on the current device: resolved once per device, with that device current.
int hi_static_scratch(mkf_ctx* c, int** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(c, e, "mkf_build_hit_index_static: cudaGetDevice");
  if (dev < 0 || dev >= HI_MAX_DEVICES) return fail(c, MKF_UNSUPPORTED, "mkf_build_hit_index_static: device ordinal >= 64");
  int* p = g_hi_static_ptr[dev].load(std::memory_order_acquire);
  if (!p) {
    e = cudaGetSymbolAddress((void**)&p, g_hi_static_scratch);
    if (e != cudaSuccess || !p) return cuda_fail(c, e, "mkf_build_hit_index_static: cudaGetSymbolAddress");
    g_hi_static_ptr[dev].store(p, std::memory_order_release);      // threads racing here store the same value
  }
  *out = p;
  return MKF_OK;
}
}  // namespace

extern "C" int mkf_build_hit_index_static(mkf_ctx* c, const mkf_hits* h, mkf_hit_index* out, void* stream) {
  if (!c) return MKF_INVALID_ARG;
  if (!h || !out || !out->bin_off || !out->sorted_id || !out->vmax || !h->layer_off)
    return fail(c, MKF_INVALID_ARG, "mkf_build_hit_index_static: null argument");
  if (h->n_events < 1 || h->n_hits < 0) return fail(c, MKF_INVALID_ARG, "mkf_build_hit_index_static: bad sizes");
  if (h->n_hits > MKF_STATIC_MAX_HITS)
    return fail(c, MKF_UNSUPPORTED, "mkf_build_hit_index_static: n_hits exceeds MKF_STATIC_MAX_HITS (1048576); use mkf_build_hit_index");
  if (h->n_hits > 0 && (!h->x || !h->y || !h->z || !h->V)) return fail(c, MKF_INVALID_ARG, "mkf_build_hit_index_static: null hit array");
  const size_t cnt_smem = (size_t)c->g.n_phi * c->g.n_eta * 4;
  if (cnt_smem > 64 * 1024)
    return fail(c, MKF_UNSUPPORTED, "mkf_build_hit_index_static: more than 16384 bins per layer; use mkf_build_hit_index");
  cudaStream_t st = (cudaStream_t)stream;
  const int nseg = h->n_events * c->g.n_layers;
  const size_t nbins = (size_t)nseg * c->g.n_phi * c->g.n_eta;
  if (h->n_hits == 0) {                                        // nothing to place: all offsets are zero
    cudaError_t e0 = cudaMemsetAsync(out->bin_off, 0, (nbins + 1) * 4, st);
    if (e0 == cudaSuccess) e0 = cudaMemsetAsync(out->vmax, 0, (size_t)nseg * 8, st);
    if (e0 != cudaSuccess) return cuda_fail(c, e0, "mkf_build_hit_index_static: memset");
    return MKF_OK;
  }
  int* scratch = nullptr;
  { const int rc = hi_static_scratch(c, &scratch); if (rc) return rc; }
  HiArgs a;
  a.hits = hits_dev(h); a.n_layers = c->g.n_layers; a.n_phi = c->g.n_phi; a.n_eta = c->g.n_eta;
  a.key = scratch; a.tmp_id = scratch + MKF_STATIC_MAX_HITS; a.cnt = nullptr;
  a.bin_off = out->bin_off; a.sorted_id = out->sorted_id; a.vmax = out->vmax; a.packed = (float4*)out->packed;
  a.mask = nullptr; a.n_bins = nbins;
  const size_t smem_s = cnt_smem + (size_t)HfSmall::tmpcap * 4, smem_l = cnt_smem + (size_t)HfLarge::tmpcap * 4;
  const bool large = (size_t)h->n_hits > (size_t)nseg * 4096;
  cudaError_t e1 = large ? cudaFuncSetAttribute(hi_fused_kernel<HfLarge>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_l)
                         : cudaFuncSetAttribute(hi_fused_kernel<HfSmall>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_s);
  if (e1 != cudaSuccess) return cuda_fail(c, e1, "mkf_build_hit_index_static: shared memory attribute");
  if (large) hi_fused_kernel<HfLarge><<<nseg, HfLarge::block, smem_l, st>>>(c->g, a);
  else hi_fused_kernel<HfSmall><<<nseg, HfSmall::block, smem_s, st>>>(c->g, a);
  MKF_LAUNCHED(c, "hi_fused_kernel");
  return MKF_OK;
}
