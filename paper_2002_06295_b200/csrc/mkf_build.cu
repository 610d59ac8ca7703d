// mkf_build.cu — a12 / C9: combinatorial track building ("combinatorial search ... from a seed in the
// innermost layers, proceeding outwards", "only the best ranking ones are cloned at each layer (with
// a per-seed cap)", PAPER.md:5 short-track preservation).
//
// Three kernels:
//   bs_seed_kernel   one thread per seed: the seed is fitted through its own three hits (U18b); its factored state
//                    goes to the workspace, its key (event, plan, eta, phi) to a counting sort;
//   (counting sort)  seeds ordered by that key, so that the seeds of a CTA walk the same layers and hit bins;
//   mkf_build_kernel one CTA = NS seeds x 8 candidate slots, candidate states in SHARED memory; per plan step the CTA
//                    goes through phases, each with every lane busy:
//       P  propagate + material + window (a2-a5): the live candidates of all seeds, compacted, one thread each;
//       S  chi2 scan (a6): the eta rows of all windows flattened into one list, SCAN_G lanes walk one row together
//          (16-byte positions of a row are contiguous; survivors of the position test read their 32-byte covariance);
//          accepted hits are appended to the candidate's short list;
//       T  top-N per seed (a8): 8 lanes of a seed (lane = parent slot) offer the head of their sorted list or their
//          miss / pass-through child, whichever ranks first under U14; shuffle tournaments pick max_cand children;
//       U  update (a7): one thread per chosen child takes its parent's propagated state from shared memory, updates
//          it with the hit, and writes the new live set back (non-finite children are dropped, R1).
//   Hit lists are a trellis in the workspace (per step and slot: hit id and parent slot); the winner's list is read
//   back at the end. Stopped candidates are offered to the seed's `best short` slot (a9), whose state lives in the
//   output arrays.
#include "mkf_ctx.h"
#include "mkf_scan.cuh"

using namespace mkf;

namespace {

constexpr int G = 8;                 // candidate slots per seed == MAX_CAND
#ifndef MKF_BUILD_NS
#define MKF_BUILD_NS 16
#endif
constexpr int NS = MKF_BUILD_NS;     // seeds per CTA
constexpr int SL = NS * G;           // candidate slots per CTA
constexpr int BT = SL;               // threads per CTA: one per slot
constexpr int LC = 8;                // accepted hits kept per candidate and layer (a seed keeps at most MAX_CAND children)
constexpr int ROWCAP = 24 * NS;        // row parts (contiguous runs of hits) in the CTA's table per scan round
constexpr int SQCAP = 48 * NS;        // survivors of the position test queued per scan pass (= hits looked at per pass)
constexpr int RUN_MAX = (1 << 22) - 1; // longest run of hits in one table entry (queue entries hold run << 22 | offset)
constexpr int NWARP = BT / 32, WQ = SQCAP / NWARP;   // survivor queue of one warp
constexpr int HIT_NONE = 0x7fffffff; // "hit id" of miss / pass-through children in the order U14
static_assert(G == MAX_CAND, "one slot per candidate");
static_assert(BT % 32 == 0 && BT <= 1024, "CTA size");

// fields of a candidate state in shared memory, [field][slot]
enum { F_X, F_Y, F_Z, F_XL, F_YL, F_ZL, F_IPT, F_PHI, F_TH, F_CPH, F_SPH, F_CTH, F_STH, F_FK, F_FCB, F_FSB, F_U0,
       F_D0 = F_U0 + 10, NF = F_D0 + 5 };
// per-seed record of the seed kernel in the workspace, [field][seed]
enum { W_CHI2 = NF, W_NH, W_LAST, W_STAT, W_OK, NW };

enum : int { FL_SCAN = 1, FL_PASS = 2, FL_MISS = 4, FL_OFFER = 8, FL_OFFER_MISS = 16 };

struct BuildArgs {
  HitsDev hits;
  const unsigned* bin_off; const int* sorted_id; const float* vmax; const float4* packed;
  int n; const float* par; const float* cov; const signed char* q; const int* seed_event; const int* seed_hits;
  const signed char* plan; int max_plan_len;
  float* par_out; float* cov_out; float* chi2; float* score; int* nhits; int* nmiss; int* hit_ids; unsigned* status;
  float* wseed;             // [NW][n]   seed kernel -> build kernel
  unsigned* trellis;        // [n][mpl][G]
  int* trellis2;            // [n][mpl][G] R15: second hit of a step (-2: none); null without overlap recovery
  int* hit_ids2;            // [mpl][n] or null
  const int* order;         // [n] seed processed at position k
  unsigned* key; unsigned* bucket; int n_buckets;      // counting sort of the seeds
  unsigned long long* counters;
};

struct Smem {
  float A[NF][SL];          // live candidates as they stand before this layer
  float B[NF][SL];          // the same candidates propagated to this layer (material applied)
  float chi2[SL]; int cnt[SL];                     // cnt = nhits | nmiss << 8 | consec << 16
  float tt[SL], tz[SL], zz[SL], lim1[SL], lim2[SL];          // lim = (variance bound of the residual) x 1.0001: r^2 > cut x lim rejects
  int flag[SL]; unsigned ostat[SL];
  uint2 rows[ROWCAP]; int n_rows, more;                       // runs of hits to scan: (slot | n << 8, first position); more: a window has rows left
  int runpre[ROWCAP + 1];                                     // exclusive prefix of the runs' lengths: the hits of a round as one list
  unsigned sq[SQCAP + BT]; int next;                            // survivors of the position test: run << 22 | offset in the run
  int wrow[SL], wphi[SL];                                     // window: next row | end row << 8 ; w0 | wn << 8
  unsigned long long lkey[LC][SL];                 // the LC best hits of the candidate on this layer, ascending:
                                                   // chi2 bits << 32 | position t of the hit in the sorted index
  int sel[SL], sel_t[SL], sel_hit[SL], sel_hit2[SL];  // the children picked for the new live set: parent | kind << 3 | dead << 8
  int plist[SL]; int nP;
  int wsum[BT / 32];
  int n_live[NS], p0[NS], plen[NS], ev[NS], last[NS], seed[NS];
  float aq[NS];
};

static_assert((sizeof(Smem) + 1024) * (64 / NS) <= 228 * 1024, "64 seeds per SM");

__device__ __forceinline__ float score_of(const ParamsDev& p, int nh, int nm, float chi2) {
  return p.score_hit * (float)nh - p.score_miss * (float)nm - chi2;
}

__device__ __forceinline__ void st_state(float (*M)[SL], int slot, const KState& S) {
  M[F_X][slot] = S.x; M[F_Y][slot] = S.y; M[F_Z][slot] = S.z; M[F_XL][slot] = S.xl; M[F_YL][slot] = S.yl; M[F_ZL][slot] = S.zl;
  M[F_IPT][slot] = S.ipt; M[F_PHI][slot] = S.phi; M[F_TH][slot] = S.th;
  M[F_CPH][slot] = S.cph; M[F_SPH][slot] = S.sph; M[F_CTH][slot] = S.cth; M[F_STH][slot] = S.sth;
  M[F_FK][slot] = __int_as_float(S.f.kind); M[F_FCB][slot] = S.f.cb; M[F_FSB][slot] = S.f.sb;
#pragma unroll
  for (int k = 0; k < 10; k++) M[F_U0 + k][slot] = S.u[k];
#pragma unroll
  for (int k = 0; k < 5; k++) M[F_D0 + k][slot] = S.d[k];
}
__device__ __forceinline__ void ld_state(const float (*M)[SL], int slot, KState& S) {
  S.x = M[F_X][slot]; S.y = M[F_Y][slot]; S.z = M[F_Z][slot]; S.xl = M[F_XL][slot]; S.yl = M[F_YL][slot]; S.zl = M[F_ZL][slot];
  S.ipt = M[F_IPT][slot]; S.phi = M[F_PHI][slot]; S.th = M[F_TH][slot];
  S.cph = M[F_CPH][slot]; S.sph = M[F_SPH][slot]; S.cth = M[F_CTH][slot]; S.sth = M[F_STH][slot];
  S.f.kind = __float_as_int(M[F_FK][slot]); S.f.cb = M[F_FCB][slot]; S.f.sb = M[F_FSB][slot];
#pragma unroll
  for (int k = 0; k < 10; k++) S.u[k] = M[F_U0 + k][slot];
#pragma unroll
  for (int k = 0; k < 5; k++) S.d[k] = M[F_D0 + k][slot];
}

// asinh to ~1e-6 absolute for |x| up to e^4 (one lg2.approx, one rsqrt-based sqrt): the eta edges of the window carry
// a margin of 2e-5 + 1e-5 |eta| below
__device__ __forceinline__ float window_asinh(float x) {
  const float ax = fabsf(x);
  return copysignf(fast_log(ax + good_sqrt(fmaf(ax, ax, 1.f))), x);
}

// U11: window of bins that contains every hit with chi2 < cut.
__device__ __forceinline__ void window(const GeomDev& g, const LayerDev& L, float cut, const KState& S,
                                       float tt, float zz_or_yy, float vxy, float vzz, int& e0, int& e1, int& p0, int& np) {
  const float x = S.x + S.xl, y = S.y + S.yl, z = S.z + S.zl;
  const float php = atan2f(y, x);
  float dphi, eta_a, eta_b;
  if (L.kind == 0) {
    const float R = L.pos;
    const float dz = sqrtf(cut * (zz_or_yy + vzz));
    const float a1 = sqrtf(cut * (fmaxf(tt, 0.f) + vxy)) / R;
    const float a2 = sqrtf(cut * vxy) / R + 2e-6f;
    dphi = a2 < 2.f ? acosf(1.f - a2) : PI_F;
    if (a1 < 1.f && dphi <= 0.5f * PI_F) dphi = fminf(dphi, asinf(a1));
    eta_a = window_asinh((z - dz) / R); eta_b = window_asinh((z + dz) / R);
  } else {
    const float r = sqrtf(fmaf(x, x, y * y));
    const float rw = sqrtf(cut * (fmaxf(tt + zz_or_yy, 0.f) + vxy)) * (1.f + 1e-5f);
    dphi = rw < r ? asinf(rw / r) : PI_F;
    const float rlo = fmaxf(r - rw, 1e-3f), rhi = r + rw;
    const float ea = window_asinh(L.pos / rlo), eb = window_asinh(L.pos / rhi);
    eta_a = fminf(ea, eb); eta_b = fmaxf(ea, eb);
  }
  // The (dphi, eta) box is already a proven superset of {chi2 < cut} (U11); it only needs margins for the fp32
  // evaluation of its edges against the fp64 bin keys of the hits (C8), not whole extra bins.
  dphi = dphi * (1.f + 1e-4f) + 2e-5f;
  const float esc = fast_div((float)g.n_eta, L.eta_hi - L.eta_lo);
  const float em = 2e-5f + 1e-5f * fmaxf(fabsf(eta_a), fabsf(eta_b));
  int ia = (int)floorf((eta_a - em - L.eta_lo) * esc), ib = (int)floorf((eta_b + em - L.eta_lo) * esc);
  e0 = min(max(ia, 0), g.n_eta - 1); e1 = min(max(ib, 0), g.n_eta - 1);
  if (!(dphi < PI_F)) { p0 = 0; np = g.n_phi; return; }
  const float ibw = (float)g.n_phi * (1.f / (2.f * PI_F));
  const int a = (int)floorf((php - dphi + PI_F) * ibw);
  const int b = (int)floorf((php + dphi + PI_F) * ibw);
  const int cnt = b - a + 1;
  if (cnt >= g.n_phi) { p0 = 0; np = g.n_phi; return; }
  p0 = a < 0 ? a + g.n_phi : (a >= g.n_phi ? a - g.n_phi : a); np = cnt;          // dphi < pi: a in (-n_phi, 2 n_phi)
}

// ---- seed phase -----------------------------------------------------------------------------------------------
// One thread per seed: fit through its own three hits (U18b). Writes the factored state and the bookkeeping to the
// workspace, the fallback output (the seed candidate itself, C9 last line) to the output arrays, the seed's hits to
// slot 0 of its trellis, and its sort key.
__global__ void __launch_bounds__(128) bs_seed_kernel(const __grid_constant__ GeomDev g, const __grid_constant__ ParamsDev p,
                                                      const __grid_constant__ BuildArgs a) {
  const int i = blockIdx.x * 128 + threadIdx.x;
  if (i >= a.n) return;
  const size_t n = (size_t)a.n;
  const int mpl = a.max_plan_len;
  unsigned* tr = a.trellis + (size_t)i * mpl * G;
  const int pl = a.plan[i], ev = a.seed_event[i];
  float chi2 = 0.f; int nh = 0, last_step = -1; unsigned stat = 0; bool ok = true;
  KState S;
  load_params(S, a.par, n, (size_t)i);
  bool has_ud = false;
  int p0 = 0, plen = 0;
  if ((unsigned)pl >= (unsigned)g.n_plans || (unsigned)ev >= (unsigned)a.hits.n_events) { stat |= ST_TRUNC; ok = false; }
  else {
    p0 = g.plan_off[pl];
    plen = min(g.plan_off[pl + 1] - p0, mpl);
    const float qk = -(float)a.q[i] * KAPPA;
    const int* loff = a.hits.layer_off + (size_t)ev * (g.n_layers + 1);
    for (int k = 0; k < 3 && ok; k++) {
      const int hid = a.seed_hits[(size_t)k * n + i];
      int lay = -1;
      for (int l = 0; l < g.n_layers; l++) if (hid >= loff[l] && hid < loff[l + 1]) { lay = l; break; }
      int step = -1;
      if (lay >= 0) for (int s = last_step + 1; s < plen; s++) if ((int)g.plan_layers[p0 + s] == lay) { step = s; break; }
      if (step < 0) { stat |= ST_TRUNC; ok = false; break; }
      const LayerDev& L = g.layers[lay];
      const unsigned rc = step_to_layer(S, !has_ud, a.cov, n, (size_t)i, L, qk * g.bz_layer[lay], p.graze_cos_min, p.material_flags, false);
      if (rc) { stat |= rc; ok = false; break; }
      has_ud = true;
      Hit H; load_hit(H, a.hits, hid);
      SInv o; float c2;
      hit_to_local(S, H, o);
      if (!kalman_update(S, o, c2)) { stat |= ST_S_NOT_PD; ok = false; break; }
      for (int s = last_step + 1; s < step; s++) tr[s * G] = 0u;            // hit code 0 == -2 (not crossed), parent 0
      if (a.trellis2) for (int s = last_step + 1; s <= step; s++) a.trellis2[((size_t)i * mpl + s) * G] = -2;
      chi2 += c2; nh++; last_step = step;
      tr[step * G] = (unsigned)(hid + 2);
    }
  }
  if (has_ud) store_state(S, a.par_out, a.cov_out, n, (size_t)i);
  else copy_seed(a.par, a.cov, a.par_out, a.cov_out, n, (size_t)i);
  float* w = a.wseed + i;
  w[(size_t)F_X * n] = S.x; w[(size_t)F_Y * n] = S.y; w[(size_t)F_Z * n] = S.z;
  w[(size_t)F_XL * n] = S.xl; w[(size_t)F_YL * n] = S.yl; w[(size_t)F_ZL * n] = S.zl;
  w[(size_t)F_IPT * n] = S.ipt; w[(size_t)F_PHI * n] = S.phi; w[(size_t)F_TH * n] = S.th;
  w[(size_t)F_CPH * n] = S.cph; w[(size_t)F_SPH * n] = S.sph; w[(size_t)F_CTH * n] = S.cth; w[(size_t)F_STH * n] = S.sth;
  w[(size_t)F_FK * n] = __int_as_float(S.f.kind); w[(size_t)F_FCB * n] = S.f.cb; w[(size_t)F_FSB * n] = S.f.sb;
#pragma unroll
  for (int k = 0; k < 10; k++) w[(size_t)(F_U0 + k) * n] = S.u[k];
#pragma unroll
  for (int k = 0; k < 5; k++) w[(size_t)(F_D0 + k) * n] = S.d[k];
  w[(size_t)W_CHI2 * n] = chi2; w[(size_t)W_NH * n] = __int_as_float(nh); w[(size_t)W_LAST * n] = __int_as_float(last_step);
  w[(size_t)W_STAT * n] = __int_as_float((int)stat); w[(size_t)W_OK * n] = __int_as_float(ok ? 1 : 0);
  // sort key: seeds that will walk the same layers and bins next to each other (any order gives the same tracks)
  const float x = S.x + S.xl, y = S.y + S.yl;
  int ip = (int)((atan2f(y, x) + PI_F) * (16.f / (2.f * PI_F))); ip = min(max(ip, 0), 15);
  int ie = (int)((S.cth + 1.f) * 8.f); ie = min(max(ie, 0), 15);          // cos(theta) is monotone in eta
  const int pe = ok ? ((ev * g.n_plans + pl) * 16 + ie) * 16 + ip : a.n_buckets - 1;       // failed seeds last
  a.key[i] = (unsigned)pe;
  atomicAdd(&a.bucket[pe], 1u);
}

__global__ void __launch_bounds__(256) bs_order_kernel(int n, const unsigned* __restrict__ key, unsigned* cursor, int* order) {
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i >= n) return;
  order[atomicAdd(&cursor[key[i]], 1u)] = i;
}

// ---- the chi2 of one hit against one propagated candidate; appends accepted hits to the candidate's list ---------
struct ScanCand { float x, y, z, xl, yl, zl, cb, sb, tt, tz, zz, lim1, lim2; int kind; };

constexpr unsigned long long KEY_NONE = ~0ull;

// Keeps the nk (<= LC) smallest keys of a candidate, sorted, under concurrent insertion by any lanes of the CTA: the key
// sinks through the list by atomic minima, each position keeping the smaller key and handing the larger one down.
// Whatever the interleaving, position k ends up with the minimum of everything offered to it, i.e. the (k+1)-th
// smallest key. The last position only ever decreases, so a key that is not below it can be dropped without an atomic.
__device__ __forceinline__ void accept_hit(Smem& sm, int slot, int nk, float c2, unsigned t) {
  unsigned long long key = ((unsigned long long)__float_as_uint(fmaxf(c2, 0.f)) << 32) | t;
  if (key >= sm.lkey[nk - 1][slot]) return;
#pragma unroll 1
  for (int k = 0; k < nk; k++) {
    const unsigned long long old = atomicMin(&sm.lkey[k][slot], key);
    if (old == KEY_NONE) break;                                    // took an empty place
    if (old > key) key = old;                                      // displaced a larger key: it sinks further
  }
}

__device__ __forceinline__ void load_scan_cand(const Smem& sm, int slot, ScanCand& c) {
  c.x = sm.B[F_X][slot]; c.y = sm.B[F_Y][slot]; c.z = sm.B[F_Z][slot];
  c.xl = sm.B[F_XL][slot]; c.yl = sm.B[F_YL][slot]; c.zl = sm.B[F_ZL][slot];
  c.kind = __float_as_int(sm.B[F_FK][slot]); c.cb = sm.B[F_FCB][slot]; c.sb = sm.B[F_FSB][slot];
  c.tt = sm.tt[slot]; c.tz = sm.tz[slot]; c.zz = sm.zz[slot]; c.lim1 = sm.lim1[slot]; c.lim2 = sm.lim2[slot];
}

// U14 as two integer keys, smaller = ranks first: k1 = (score descending, chi2 ascending), k2 = (parent, hit), the hit
// given by its position in the sorted index (bin, then id; misses last): reading R11 of DESIGN.md
__device__ __forceinline__ unsigned long long rank_key1(float score, float chi2) {
  unsigned su = __float_as_uint(score);
  su = (su & 0x80000000u) ? ~su : (su | 0x80000000u);            // ascending in the float order
  return ((unsigned long long)(~su) << 32) | __float_as_uint(chi2);
}
__device__ __forceinline__ unsigned rank_key2(int parent, int hit) { return ((unsigned)parent << 28) | ((unsigned)hit & 0x0fffffffu); }
// R15: one more hit of the layer from an overlapping module. S: the child's state, already
// updated with its first hit (position t1 in the sorted index, module mod1). Candidates: the parent's list of this layer
// (its max_cand best hits by chi2 against the propagated state) behind the first hit. The best chi2 against S below the cut wins; the update
// is taken only if it stays finite. Returns the hit id taken (or -2) and adds its chi2. Kept out of line: it is off the
// path of the plain build.
__device__ __noinline__ int overlap_hit(const BuildArgs& a, const ParamsDev& p, const Smem& sm, int ps, unsigned t1, int mod1,
                                        KState& S, float& chi2_add) {
  float tt, tz, zz;
  cov_aa(S, tt, tz, zz);
  float best = p.chi2_cut; int best_id = -2; Hit Hb;
  bool after = false;                                              // only hits that rank after the first one in the list
  for (int k = 0; k < p.max_cand; k++) {
    const unsigned long long key = sm.lkey[k][ps];
    if (key == KEY_NONE) break;
    const unsigned t2 = (unsigned)key;
    if (t2 == t1) { after = true; continue; }
    if (!after) continue;
    Hit H2; int id2, mod2;
    if (a.packed) {
      const float4 q0 = __ldg(a.packed + t2);
      const float4* cv = a.packed + packed_cov_off(a.hits.n_hits) + (size_t)2 * t2;
      const float4 b = __ldg(cv), d = __ldg(cv + 1);
      H2.x = q0.x; H2.y = q0.y; H2.z = q0.z; id2 = __float_as_int(q0.w); mod2 = __float_as_int(d.z);
      H2.v[0] = b.x; H2.v[1] = b.y; H2.v[2] = b.z; H2.v[3] = b.w; H2.v[4] = d.x; H2.v[5] = d.y;
    } else { id2 = a.sorted_id[t2]; mod2 = a.hits.module[id2]; load_hit(H2, a.hits, id2); }
    if (mod2 == mod1) continue;
    SInv o2; float c2b;
    if (!chi2_local(S, tt, tz, zz, H2, o2, c2b)) continue;
    if (c2b < best) { best = c2b; best_id = id2; Hb = H2; }
  }
  if (best_id < 0) return -2;
  KState S2 = S;
  SInv o; float c2u;
  hit_to_local(S2, Hb, o);
  if (!(kalman_update(S2, o, c2u) && state_finite(S2) && fabsf(c2u) <= 3.0e38f)) return -2;
  S = S2; chi2_add = c2u;
  return best_id;
}

// The state of a slot written to the output arrays (offers to `best short`, final readout): one copy of the U D U^T
// expansion and the rotation to the global frame for its three call sites, out of the layer loop's instruction footprint.
__device__ __noinline__ void store_slot_state(const float (*M)[SL], int slot, float* par_out, float* cov_out, size_t n, size_t i) {
  KState S; ld_state(M, slot, S);
  store_state(S, par_out, cov_out, n, i);
}

#ifndef MKF_BUILD_MIN_BLOCKS
#define MKF_BUILD_MIN_BLOCKS (64 / MKF_BUILD_NS)
#endif
template <bool COUNT, bool PACKED>
__global__ void __launch_bounds__(BT, MKF_BUILD_MIN_BLOCKS) mkf_build_kernel(const __grid_constant__ GeomDev g,
                                                                const __grid_constant__ ParamsDev p,
                                                                const __grid_constant__ BuildArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int sl = tid >> 3;                                   // seed of this thread's group (phases T, offers)
  const int sub = tid & (G - 1);                             // candidate slot inside the seed
  const int gbase = lane & ~(G - 1);
  const unsigned gm = 0xffu << gbase;
  const size_t n = (size_t)a.n;
  const int mpl = a.max_plan_len;
  const int nb = g.n_phi * g.n_eta;
  unsigned n_steps = 0, n_pos = 0, n_c2 = 0, n_acc = 0, n_upd = 0, n_rowt = 0, n_rowo = 0;        // COUNT only

  // ---- load the seeds of this CTA ------------------------------------------------------------------------------
  const int pos = blockIdx.x * NS + sl;
  const int i = pos < a.n ? a.order[pos] : -1;                // the seed of this thread's group
  float seed_chi2 = 0.f; int seed_nh = 0, seed_last = -1; unsigned seed_stat = 0; bool seed_ok = false;
  if (i >= 0) {
    const float* w = a.wseed + i;
    seed_chi2 = w[(size_t)W_CHI2 * n]; seed_nh = __float_as_int(w[(size_t)W_NH * n]); seed_last = __float_as_int(w[(size_t)W_LAST * n]);
    seed_stat = (unsigned)__float_as_int(w[(size_t)W_STAT * n]); seed_ok = __float_as_int(w[(size_t)W_OK * n]) != 0;
    if (sub == 0) {
      int p0 = 0, plen = 0;
      if (seed_ok) { const int pl = a.plan[i]; p0 = g.plan_off[pl]; plen = min(g.plan_off[pl + 1] - p0, mpl); }
      sm.p0[sl] = p0; sm.plen[sl] = plen; sm.ev[sl] = seed_ok ? a.seed_event[i] : 0; sm.last[sl] = seed_last; sm.seed[sl] = i;
      sm.aq[sl] = -(float)a.q[i] * KAPPA;                     // times Bz of the step (R13)
      sm.n_live[sl] = seed_ok ? 1 : 0;
      if (seed_ok) {
#pragma unroll
        for (int k = 0; k < NF; k++) sm.A[k][tid] = w[(size_t)k * n];
        sm.chi2[tid] = seed_chi2; sm.cnt[tid] = seed_nh;
      }
    }
  } else if (sub == 0) { sm.n_live[sl] = 0; sm.plen[sl] = 0; sm.last[sl] = -1; sm.seed[sl] = -1; sm.p0[sl] = 0; sm.ev[sl] = 0; sm.aq[sl] = 0.f; }
  unsigned* trellis = a.trellis + (size_t)(i >= 0 ? i : 0) * mpl * G;

  // best short candidate of the seed (replicated in the 8 lanes of the group)
  bool bs_have = false; float bs_score = 0.f, bs_chi2 = 0.f; int bs_nh = 0, bs_nm = 0, bs_step = 0, bs_parent = 0, bs_last = -2;
  unsigned bs_stat = 0;
  int t_last = seed_last;                                    // last step at which the live set was rewritten
  __syncthreads();

  for (int s = 0; s < mpl; s++) {
    // The rows of a window go to the CTA's table as runs of hits, with their bin offsets (the next row's are fetched
    // ahead). A window that finds the table full keeps its place and goes on in the next scan round.
    auto push_rows = [&](int slot) {
      const int ssl = slot >> 3;
      const int lay = g.plan_layers[sm.p0[ssl] + s];
      int ie = sm.wrow[slot] & 0xff; const int iend = sm.wrow[slot] >> 8;
      if (ie >= iend) return;
      const int w0 = sm.wphi[slot] & 0xff, wn = sm.wphi[slot] >> 8;
      const unsigned* row = a.bin_off + ((size_t)sm.ev[ssl] * g.n_layers + lay) * (size_t)nb + ie * g.n_phi;
      const int wend = min(w0 + wn, g.n_phi), wrap = w0 + wn - g.n_phi;
      unsigned tb0 = __ldg(row + w0), te0 = __ldg(row + wend), tb1 = 0, te1 = 0;
      if (wrap > 0) { tb1 = __ldg(row); te1 = __ldg(row + wrap); }
      for (; ie < iend; ie++) {
        const unsigned cb0 = tb0, ce0 = te0, cb1 = tb1, ce1 = te1;
        if (ie + 1 < iend) {
          row += g.n_phi;
          tb0 = __ldg(row + w0); te0 = __ldg(row + wend);
          if (wrap > 0) { tb1 = __ldg(row); te1 = __ldg(row + wrap); }
        }
        // one entry per non-empty part; a run longer than RUN_MAX hits (never met in practice) goes in as several
        const unsigned n0 = ce0 - cb0, n1 = ce1 > cb1 ? ce1 - cb1 : 0u;
        const bool lng = n0 > (unsigned)RUN_MAX || n1 > (unsigned)RUN_MAX;
        const int np = lng ? (int)((n0 + RUN_MAX - 1) / RUN_MAX + (n1 + RUN_MAX - 1) / RUN_MAX) : (n0 ? 1 : 0) + (n1 ? 1 : 0);
        if (np == 0) continue;
        const int k = atomicAdd(&sm.n_rows, np);
        if (COUNT) n_rowt += np;
        if (k + np > ROWCAP) {                                // no room: this row and the ones behind it wait for the next round
          for (int kk = k; kk < min(k + np, ROWCAP); kk++) sm.rows[kk] = make_uint2((unsigned)slot, 0u);
          sm.more = 1;
          if (COUNT) n_rowo += np;
          break;
        }
        if (!lng) {
          if (n0) sm.rows[k] = make_uint2((unsigned)slot | (n0 << 8), cb0);
          if (n1) sm.rows[k + (n0 ? 1 : 0)] = make_uint2((unsigned)slot | (n1 << 8), cb1);
        } else {
          int kk = k;
#pragma unroll 1
          for (unsigned o = 0; o < n0; o += RUN_MAX) sm.rows[kk++] = make_uint2((unsigned)slot | (min(n0 - o, (unsigned)RUN_MAX) << 8), cb0 + o);
#pragma unroll 1
          for (unsigned o = 0; o < n1; o += RUN_MAX) sm.rows[kk++] = make_uint2((unsigned)slot | (min(n1 - o, (unsigned)RUN_MAX) << 8), cb1 + o);
        }
      }
      sm.wrow[slot] = ie | (iend << 8);
    };
    // ---- which slots propagate at this step: compacted list over the CTA ------------------------------------------
    const int nl_prev = sm.n_live[sl];
    const bool seed_act = i >= 0 && seed_ok && s > seed_last && s < sm.plen[sl] && nl_prev > 0;     // uniform in the group
    const bool parent_live = seed_act && sub < nl_prev;
    {
      const unsigned bal = __ballot_sync(0xffffffffu, parent_live);
      if (lane == 0) sm.wsum[warp] = __popc(bal);
      sm.flag[tid] = 0; sm.wrow[tid] = 0;
      if (tid == 0) { sm.n_rows = 0; sm.more = 0; }
#pragma unroll
      for (int k = 0; k < LC; k++) sm.lkey[k][tid] = KEY_NONE;
      __syncthreads();
      int base = 0, tot = 0;
#pragma unroll
      for (int w2 = 0; w2 < BT / 32; w2++) { const int c = sm.wsum[w2]; if (w2 < warp) base += c; tot += c; }
      if (tot == 0) {                                         // no seed of this CTA is active at this step
        __syncthreads();
        continue;
      }
      if (parent_live) sm.plist[base + __popc(bal & ((1u << lane) - 1u))] = tid;
      if (tid == 0) sm.nP = tot;
      __syncthreads();
    }

    // ---- phase P: propagate, material, window ---------------------------------------------------------------------
    if (tid < sm.nP) {
      const int slot = sm.plist[tid];
      const int ssl = slot >> 3;
      const int lay = g.plan_layers[sm.p0[ssl] + s];
      const LayerDev& L = g.layers[lay];
      KState S; ld_state(sm.A, slot, S);
      Prop P;
      const unsigned rc = propagate_geom(S, L, sm.aq[ssl] * g.bz_layer[lay], p.graze_cos_min, p.material_flags, true, P);
      const int cn = sm.cnt[slot];
      const int nh = cn & 0xff, consec = cn >> 16;
      if (rc & (ST_UNREACH | ST_SKIP_ACC)) {
        sm.flag[slot] = FL_PASS;                              // silent skip: competes unchanged (C9.1)
      } else if (rc) {                                        // grazing / energy exhausted: the candidate stops
        if (nh >= p.min_hits_keep) { sm.flag[slot] = FL_OFFER; sm.ostat[slot] = rc; }
      } else {
        commit_step(S, P, p.material_flags);
        if (COUNT) n_steps++;
        st_state(sm.B, slot, S);
        float tt, tz, zz;
        cov_aa(S, tt, tz, zz);
        const size_t seg = (size_t)sm.ev[ssl] * g.n_layers + lay;
        const float vxy = a.vmax[2 * seg], vzz = a.vmax[2 * seg + 1];
        int e0, e1, w0, wn;
        window(g, L, p.chi2_cut, S, tt, zz, vxy, vzz, e0, e1, w0, wn);
        sm.tt[slot] = tt; sm.tz[slot] = tz; sm.zz[slot] = zz;
        sm.lim1[slot] = (tt + vxy) * 1.0001f;
        sm.lim2[slot] = (zz + (L.kind == 0 ? vzz : vxy)) * 1.0001f;
        sm.wrow[slot] = e0 | ((e1 + 1) << 8); sm.wphi[slot] = w0 | (wn << 8);     // its rows go to the table below
        int fl = FL_SCAN;
        // miss child (C9.5): stopped if it reaches the consecutive-miss limit
        if (consec + 1 >= p.max_consec_miss) { if (nh >= p.min_hits_keep) { fl |= FL_OFFER_MISS; sm.ostat[slot] = 0; } }
        else fl |= FL_MISS;
        sm.flag[slot] = fl;
      }
    }

    // ---- phase S: the hits of all runs of the table as ONE list. Pass A: every thread takes an equal share of it and
    // tests positions (16 B per hit); the survivors go to a queue. Pass B: one thread per queued survivor reads the
    // covariance (32 B) and evaluates chi2; accepted hits sink into their candidate's list. Both passes run with every
    // lane busy whatever the sizes of the windows. Further rounds while windows have rows left. --------------------------
    for (bool round0 = true;; round0 = false) {
      if (!round0) {
        __syncthreads();
        if (tid == 0) { sm.n_rows = 0; sm.more = 0; }
        __syncthreads();
      }
      if (tid < sm.nP) push_rows(sm.plist[tid]);              // the thread that propagated the slot (no barrier needed before)
      __syncthreads();
      const int NR = min(sm.n_rows, ROWCAP);
      const int more = sm.more;
      // exclusive prefix of the run lengths
      {
        constexpr int PER = (ROWCAP + BT - 1) / BT;
        int loc[PER]; int sum = 0;
#pragma unroll
        for (int k = 0; k < PER; k++) { const int j = tid * PER + k; loc[k] = j < NR ? (int)(sm.rows[j].x >> 8) : 0; sum += loc[k]; }
        int inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int t2 = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t2; }
        if (lane == 31) sm.wsum[warp] = inc;
        __syncthreads();
        int base = 0, tot = 0;
#pragma unroll
        for (int w2 = 0; w2 < BT / 32; w2++) { const int c = sm.wsum[w2]; if (w2 < warp) base += c; tot += c; }
        int run = base + inc - sum;
#pragma unroll
        for (int k = 0; k < PER; k++) { const int j = tid * PER + k; if (j <= NR) sm.runpre[j] = run; run += loc[k]; }
        if (tid == 0) { sm.runpre[NR] = tot; sm.next = NWARP * WQ; }
        __syncthreads();
      }
      const int H = sm.runpre[NR];
      // the warps take parts of WQ hits from the list as they get free and work through them on their own: no CTA barrier
      // and no shared counter between the two passes
      unsigned* wq = sm.sq + warp * (WQ + 32);
      int nq = 0;                                             // queued survivors (uniform in the warp); a rest < 32 waits for the next part
      const unsigned lt = (1u << lane) - 1u;
      // a list of up to NWARP x WQ hits is dealt out in equal parts; of a longer one every warp gets a first part of WQ hits
      // and takes further ones from a counter as it gets free
      const int part = min(WQ, (H + NWARP - 1) / NWARP);
      const bool steal = H > NWARP * WQ;                      // sm.next starts at NWARP x WQ
      bool first = true;
      for (bool last = false; !last;) {
        int c0 = warp * part;
        if (!first) {
          if (steal) { if (lane == 0) c0 = atomicAdd(&sm.next, WQ); c0 = __shfl_sync(0xffffffffu, c0, 0); }
          else c0 = H;
        }
        first = false;
        last = c0 >= H;
        // ---- pass A: hits [c0, c1), a contiguous share per lane (its next position is fetched ahead); the loop is uniform
        // in the warp, survivors are queued by ballot -----------------------------------------------------------------
        const int c1 = min(c0 + part, H);
        const int share = last ? 0 : (c1 - c0 + 31) >> 5;
        int q = c0 + lane * share;
        const int qe = min(q + share, c1);
        int j = 0, rb = 0, re = 0, slot = 0, kind = 0;
        float cx = 0.f, cy = 0.f, cz = 0.f, cxl = 0.f, cyl = 0.f, czl = 0.f, cb = 0.f, sb = 0.f, l1 = 0.f, l2 = 0.f;
        const unsigned* worst = nullptr; const float4* pp = nullptr; float4 qn = make_float4(0.f, 0.f, 0.f, 0.f), qn2 = qn;
        if (q < qe) {
          int lo = 0, hi = NR;                                // run of hit q: last j with runpre[j] <= q
          while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (sm.runpre[mid] <= q) lo = mid; else hi = mid; }
          j = lo - 1; re = q;                                 // the first iteration opens run lo
        }
#pragma unroll 1
        for (int it = 0; it < share; it++) {
          bool surv = false; unsigned ent = 0;
          if (q < qe) {
            if (q >= re) {                                    // next run (runs of length 0 are skipped)
              do { j++; rb = sm.runpre[j]; re = sm.runpre[j + 1]; } while (q >= re);
              const uint2 r = sm.rows[j];
              slot = (int)(r.x & 0xffu);
              if (PACKED) {
                cx = sm.B[F_X][slot]; cy = sm.B[F_Y][slot]; cz = sm.B[F_Z][slot];
                cxl = sm.B[F_XL][slot]; cyl = sm.B[F_YL][slot]; czl = sm.B[F_ZL][slot];
                kind = __float_as_int(sm.B[F_FK][slot]); cb = sm.B[F_FCB][slot]; sb = sm.B[F_FSB][slot];
                l1 = sm.lim1[slot]; l2 = sm.lim2[slot];
                worst = reinterpret_cast<const unsigned*>(&sm.lkey[p.max_cand - 1][slot]) + 1;    // chi2 bits of the list's last hit
                pp = a.packed + r.y + (q - rb);
                qn = __ldg(pp);
                if (q + 1 < min(qe, re)) qn2 = __ldg(pp + 1);
              }
            }
            ent = ((unsigned)j << 22) | (unsigned)(q - rb);
            if (COUNT) n_pos++;
            if (PACKED) {
              // position first: chi2 >= (e.r)^2 / (e^T S e) for the unit vectors e = w1, w2 (Cauchy-Schwarz, U11); once
              // the candidate's list is full only a hit better than its last one can matter, so the cut follows it
              const float4 q0 = qn;
              qn = qn2;
              pp++;
              if (q + 2 < min(qe, re)) qn2 = __ldg(pp + 1);   // the hits two positions ahead of their use
              const float cut = fminf(p.chi2_cut, __uint_as_float(min(*(volatile const unsigned*)worst, 0x7f800000u)));
              const float rx = (q0.x - cx) - cxl, ry = (q0.y - cy) - cyl, rz = (q0.z - cz) - czl;
              const float r1 = kind == 0 ? cb * ry - sb * rx : rx, r2 = kind == 0 ? rz : ry;
              surv = !(r1 * r1 > cut * l1 || r2 * r2 > cut * l2);
            } else surv = true;
            q++;
          }
          const unsigned bal = __ballot_sync(0xffffffffu, surv);
          if (surv) wq[nq + __popc(bal & lt)] = ent;
          nq += __popc(bal);
        }
        __syncwarp();
        // ---- pass B: one lane per survivor, full warps only while more hits follow ----------------------------------------
        const int nproc = last ? nq : (nq & ~31);
        float4 nq0 = make_float4(0.f, 0.f, 0.f, 0.f), nb4 = nq0, nd4 = nq0; int nslot = 0; unsigned nt = 0;
        auto fetch = [&](int k) {                             // the survivor's hit, one queue entry ahead of its use
          const unsigned e = wq[k];
          const uint2 r = sm.rows[e >> 22];
          nslot = (int)(r.x & 0xffu);
          nt = r.y + (e & 0x3fffffu);
          if (PACKED) {
            nq0 = __ldg(a.packed + nt);
            const float4* cv = a.packed + packed_cov_off(a.hits.n_hits) + (size_t)2 * nt;
            nb4 = __ldg(cv); nd4 = __ldg(cv + 1);
          }
        };
        if (lane < nproc) fetch(lane);
#pragma unroll 1
        for (int k = lane; k < nproc; k += 32) {
          const int slot2 = nslot; const unsigned t = nt;
          Hit H2;
          if (PACKED) {
            H2.x = nq0.x; H2.y = nq0.y; H2.z = nq0.z;
            H2.v[0] = nb4.x; H2.v[1] = nb4.y; H2.v[2] = nb4.z; H2.v[3] = nb4.w; H2.v[4] = nd4.x; H2.v[5] = nd4.y;
          } else load_hit(H2, a.hits, a.sorted_id[t]);
          if (k + 32 < nproc) fetch(k + 32);
          ScanCand c; load_scan_cand(sm, slot2, c);
          KState Sc;                                          // only what hit_to_local / chi2_local read
          Sc.x = c.x; Sc.y = c.y; Sc.z = c.z; Sc.xl = c.xl; Sc.yl = c.yl; Sc.zl = c.zl; Sc.f.kind = c.kind; Sc.f.cb = c.cb; Sc.f.sb = c.sb;
          if (COUNT) n_c2++;
          SInv o; float c2;
          if (chi2_local(Sc, c.tt, c.tz, c.zz, H2, o, c2) && c2 < p.chi2_cut) {
            if (COUNT) n_acc++;
            accept_hit(sm, slot2, p.max_cand, c2, t);
          }
        }
        __syncwarp();
        if (!last) {
          const int rem = nq - nproc;
          const unsigned e = lane < rem ? wq[nproc + lane] : 0u;
          __syncwarp();
          if (lane < rem) wq[lane] = e;
          nq = rem;
          __syncwarp();
        }
      }
      __syncthreads();
      if (!more) break;
    }

    // ---- the lists are sorted as they stand: count this slot's entries -----------------------------------------------
    const int fl = sm.flag[tid];
    int n_hitc = 0;
    if (fl & FL_SCAN) {
#pragma unroll
      for (int k = 0; k < LC; k++) n_hitc += sm.lkey[k][tid] != KEY_NONE ? 1 : 0;
    }

    // ---- per seed group: lane = parent slot -------------------------------------------------------------------------
    const float chi2 = sm.chi2[tid];
    const int cn = sm.cnt[tid];
    const int nh = cn & 0xff, nm = (cn >> 8) & 0xff;
    // a seed all of whose candidates pass this layer by (not crossed) keeps its live set as it is
    const bool noop = seed_act && (__ballot_sync(gm, parent_live && fl != FL_PASS) & gm) == 0u;

    // offers to best_short (C9.6): first the stops found while propagating (state before the layer), then the
    // stopped miss children (propagated state), each in rank order; strict comparison with the holder
    if (seed_act && !noop) {
      const bool off0 = parent_live && (fl & FL_OFFER), off1 = parent_live && (fl & FL_OFFER_MISS);
      if (__ballot_sync(gm, off0 || off1) & gm) {
        const int onm = off1 ? nm + 1 : nm;
        float os = (off0 || off1) ? score_of(p, nh, onm, chi2) : -INFINITY, oc = chi2; int ok = (off1 ? G : 0) + sub, ol = sub;
#pragma unroll
        for (int d = 1; d < G; d <<= 1) {
          const float s2 = __shfl_xor_sync(gm, os, d), c2 = __shfl_xor_sync(gm, oc, d);
          const int k2 = __shfl_xor_sync(gm, ok, d), l2 = __shfl_xor_sync(gm, ol, d);
          const bool take = (s2 != os) ? (s2 > os) : ((c2 != oc) ? (c2 < oc) : (k2 < ok));
          if (take) { os = s2; oc = c2; ok = k2; ol = l2; }
        }
        if (!bs_have || os > bs_score || (os == bs_score && oc < bs_chi2)) {
          const int src = gbase + ol;
          if (sub == ol) store_slot_state(ok >= G ? sm.B : sm.A, tid, a.par_out, a.cov_out, n, (size_t)i);
          bs_have = true; bs_score = os; bs_chi2 = oc;
          bs_nh = __shfl_sync(gm, nh, src); bs_nm = __shfl_sync(gm, onm, src);
          bs_stat = __shfl_sync(gm, (fl & (FL_OFFER | FL_OFFER_MISS)) ? sm.ostat[tid] : 0u, src);
          bs_step = s; bs_parent = ol; bs_last = (ok >= G) ? -1 : -2;
        }
      }
    }

    // ---- phase T: top max_cand children of the seed (U14), 8-lane tournaments on integer keys -----------------------
    int my_parent = sub, n_new = 0;
    if (seed_act && !noop) {
      const float base_hit = score_of(p, nh + 1, nm, chi2);   // hit child: base_hit - c2_hit
      bool alt_avail = parent_live && (fl & (FL_MISS | FL_PASS));
      const int alt_kind = (fl & FL_MISS) ? 1 : 2;
      const unsigned long long alt_k1 = rank_key1((fl & FL_MISS) ? score_of(p, nh, nm + 1, chi2) : score_of(p, nh, nm, chi2), chi2);
      if (!parent_live) n_hitc = 0;
      int head = 0;
      int my_kind = -1, my_t = 0;
#pragma unroll 1
      for (int r = 0; r < p.max_cand; r++) {
        // head child of this lane: its next hit or its miss / pass-through child, whichever ranks first (U14)
        unsigned long long k1 = KEY_NONE; int hh = HIT_NONE, hk = 3;
        if (head < n_hitc) {
          const unsigned long long key = sm.lkey[head][tid];
          const float c2h = __uint_as_float((unsigned)(key >> 32));
          k1 = rank_key1(base_hit - c2h, chi2 + c2h); hh = (int)(unsigned)key; hk = 0;
        }
        if (alt_avail && alt_k1 < k1) { k1 = alt_k1; hh = HIT_NONE; hk = alt_kind; }     // same parent: a tie in k1 goes to the hit
        unsigned k2 = rank_key2(sub, hh);
        unsigned long long w1 = k1; unsigned w2 = k2;
#pragma unroll
        for (int d = 1; d < G; d <<= 1) {
          const unsigned long long o1 = __shfl_xor_sync(gm, w1, d); const unsigned o2 = __shfl_xor_sync(gm, w2, d);
          if (o1 < w1 || (o1 == w1 && o2 < w2)) { w1 = o1; w2 = o2; }
        }
        if (w1 == KEY_NONE) break;                            // pool exhausted (uniform in the group)
        const int wp = (int)(w2 >> 28);
        const int src = gbase + wp;
        const int wk = __shfl_sync(gm, hk, src), wh = __shfl_sync(gm, hh, src);
        if (sub == wp) { if (wk == 0) head++; else alt_avail = false; }      // the winner lane pops its head
        if (sub == r) { my_parent = wp; my_kind = wk; my_t = wh; }
        n_new = r + 1;
      }
      if (sub < n_new) { sm.sel[tid] = my_parent | (my_kind << 3); sm.sel_t[tid] = my_t; }
    }

    // ---- phase U: the chosen children, compacted over the CTA: the parent's state, updated with the hit --------------
    const bool is_child = seed_act && !noop && sub < n_new;
    {
      const unsigned bal = __ballot_sync(0xffffffffu, is_child);
      if (lane == 0) sm.wsum[warp] = __popc(bal);
      __syncthreads();
      int base = 0, tot = 0;
#pragma unroll
      for (int w2 = 0; w2 < BT / 32; w2++) { const int c = sm.wsum[w2]; if (w2 < warp) base += c; tot += c; }
      if (is_child) sm.plist[base + __popc(bal & ((1u << lane) - 1u))] = tid;
      if (tid == 0) sm.nP = tot;
      __syncthreads();
    }
    KState S;
    float c_chi2 = 0.f; int c_cnt = 0, cslot = -1, c_sel = 0, c_hit = 0, c_hit2 = -2;
    bool nan_child = false;
    if (tid < sm.nP) {
      cslot = sm.plist[tid];
      c_sel = sm.sel[cslot];
      const int kind = (c_sel >> 3) & 3;
      c_hit = kind == 1 ? -1 : -2;
      const int ps = (cslot & ~(G - 1)) + (c_sel & 7);        // parent's slot
      Hit H; int mod1 = 0;
      if (kind == 0) {                                        // the hit's record first: its latency overlaps the state loads
        if (PACKED) {
          const int t = sm.sel_t[cslot];
          const float4 q0 = __ldg(a.packed + t);
          const float4* cv = a.packed + packed_cov_off(a.hits.n_hits) + (size_t)2 * t;
          const float4 b = __ldg(cv), d = __ldg(cv + 1);
          H.x = q0.x; H.y = q0.y; H.z = q0.z; c_hit = __float_as_int(q0.w); mod1 = __float_as_int(d.z);
          H.v[0] = b.x; H.v[1] = b.y; H.v[2] = b.z; H.v[3] = b.w; H.v[4] = d.x; H.v[5] = d.y;
        } else { c_hit = a.sorted_id[sm.sel_t[cslot]]; load_hit(H, a.hits, c_hit); if (a.hit_ids2) mod1 = a.hits.module[c_hit]; }
      }
      const int pcn = sm.cnt[ps];
      c_chi2 = sm.chi2[ps];
      int c_nh = pcn & 0xff, c_nm = (pcn >> 8) & 0xff, c_consec = pcn >> 16;
      if (kind == 2) ld_state(sm.A, ps, S);                   // pass-through: the state does not move
      else ld_state(sm.B, ps, S);
      if (kind == 1) { c_nm++; c_consec++; }
      else if (kind == 0) {
        SInv o; float c2;
        hit_to_local(S, H, o);
        if (COUNT) n_upd++;
        if (kalman_update(S, o, c2) && state_finite(S) && fabsf(c2) <= 3.0e38f) {
          c_chi2 += c2; c_nh++; c_consec = 0;
          if (a.hit_ids2) {                                   // R15: one more hit from an overlapping module
            float c2b = 0.f;
            c_hit2 = overlap_hit(a, p, sm, ps, (unsigned)sm.sel_t[cslot], mod1, S, c2b);
            if (c_hit2 >= 0) { c_chi2 += c2b; c_nh++; }
          }
        } else { nan_child = true; sm.sel[cslot] = c_sel | 256; }      // dropped (C9 / R1)
      }
      c_cnt = c_nh | (c_nm << 8) | (c_consec << 16);
      sm.sel_hit[cslot] = c_hit; sm.sel_hit2[cslot] = c_hit2;  // for the trellis entries if the live set is compacted below
    }
    const bool any_nan = __syncthreads_or(nan_child);         // also: every read of A and B of this step is done
    if (any_nan) {
      // R1: the parent of a dropped child, as it stood before the layer, is offered to best_short (after the offers
      // above, in child rank order; strict comparison with the holder)
      if (seed_act && !noop) {
        const bool dead = sub < n_new && (sm.sel[tid] & 256);
        const int ps = (tid & ~(G - 1)) + my_parent;
        const int pcn = sm.cnt[ps];
        const int pnh = pcn & 0xff, pnm = (pcn >> 8) & 0xff;
        const float pchi2 = sm.chi2[ps];
        float os = (dead && pnh >= p.min_hits_keep) ? score_of(p, pnh, pnm, pchi2) : -INFINITY, oc = pchi2; int ol = sub;
#pragma unroll
        for (int d = 1; d < G; d <<= 1) {
          const float s2 = __shfl_xor_sync(gm, os, d), c2 = __shfl_xor_sync(gm, oc, d);
          const int l2 = __shfl_xor_sync(gm, ol, d);
          const bool take = (s2 != os) ? (s2 > os) : ((c2 != oc) ? (c2 < oc) : (l2 < ol));
          if (take) { os = s2; oc = c2; ol = l2; }
        }
        if (os > -INFINITY && (!bs_have || os > bs_score || (os == bs_score && oc < bs_chi2))) {
          const int src = gbase + ol;
          if (sub == ol) store_slot_state(sm.A, ps, a.par_out, a.cov_out, n, (size_t)i);
          bs_have = true; bs_score = os; bs_chi2 = oc;
          bs_nh = __shfl_sync(gm, pnh, src); bs_nm = __shfl_sync(gm, pnm, src);
          bs_stat = 0;
          bs_step = s; bs_parent = __shfl_sync(gm, my_parent, src); bs_last = -2;
        }
      }
      __syncthreads();                                        // the parents' states have been read
    }
    if (cslot >= 0 && !nan_child) {                           // the child becomes live candidate `rank` of its seed
      st_state(sm.A, cslot, S);
      sm.chi2[cslot] = c_chi2; sm.cnt[cslot] = c_cnt;
      const int si = sm.seed[cslot >> 3];
      a.trellis[((size_t)si * mpl + s) * G + (cslot & (G - 1))] = (unsigned)(c_hit + 2) | ((unsigned)(c_sel & 7) << 28);
      if (a.trellis2) a.trellis2[((size_t)si * mpl + s) * G + (cslot & (G - 1))] = c_hit2;
    }
    if (seed_act) {
      if (noop) { if (parent_live) { trellis[(size_t)s * G + sub] = (unsigned)sub << 28; if (a.trellis2) a.trellis2[((size_t)i * mpl + s) * G + sub] = -2; } }   // hit code 0 == -2 (not crossed)
      else if (sub == 0) sm.n_live[sl] = n_new;
      t_last = s;
    }
    if (any_nan) {
      // dropped children leave holes in the new live set: close them, keeping the rank order (rare)
      __syncthreads();
      if (seed_act && !noop) {
        const unsigned alive = (__ballot_sync(gm, sub < n_new && !(sm.sel[tid] & 256)) >> gbase) & 0xffu;
        if (alive != ((1u << n_new) - 1u)) {
          const int cntl = __popc(alive);
          const int srcl = sub < cntl ? (int)__fns(alive, 0, sub + 1) : sub;
          const int from = (tid & ~(G - 1)) + srcl;
          KState Sm; ld_state(sm.A, from, Sm);
          const float mchi2 = sm.chi2[from]; const int mcnt = sm.cnt[from];
          const unsigned ent = (unsigned)(sm.sel_hit[from] + 2) | ((unsigned)(sm.sel[from] & 7) << 28);
          const int ent2 = sm.sel_hit2[from];
          __syncwarp(gm);
          if (sub < cntl) {
            st_state(sm.A, tid, Sm); sm.chi2[tid] = mchi2; sm.cnt[tid] = mcnt;
            trellis[(size_t)s * G + sub] = ent;
            if (a.trellis2) a.trellis2[((size_t)i * mpl + s) * G + sub] = ent2;
          }
          if (sub == 0) sm.n_live[sl] = cntl;
        }
      }
    }
    __syncthreads();
  }

  // ---- final choice: best of live U {best_short} (C9) -----------------------------------------------------------
  if (i >= 0) {
    const int nl = sm.n_live[sl];
    const float chi2 = sm.chi2[tid];
    const int cn = sm.cnt[tid];
    const int nh = cn & 0xff, nm = (cn >> 8) & 0xff;
    const bool live = seed_ok && sub < nl;
    float fs = (live && nh >= p.min_hits_keep) ? score_of(p, nh, nm, chi2) : -INFINITY, fc = chi2; int fl2 = sub;
#pragma unroll
    for (int d = 1; d < G; d <<= 1) {
      const float s2 = __shfl_xor_sync(gm, fs, d), c2 = __shfl_xor_sync(gm, fc, d);
      const int l2 = __shfl_xor_sync(gm, fl2, d);
      const bool take = (s2 != fs) ? (s2 > fs) : ((c2 != fc) ? (c2 < fc) : (l2 < fl2));
      if (take) { fs = s2; fc = c2; fl2 = l2; }
    }
    const bool live_wins = fs > -INFINITY && !(bs_have && (bs_score > fs || (bs_score == fs && bs_chi2 < fc)));
    float o_chi2, o_score; int o_nh, o_nm, bt_step, bt_slot, tail_step = -1, tail_val = -2; unsigned o_stat;
    if (live_wins) {
      const int src = gbase + fl2;
      if (sub == fl2) store_slot_state(sm.A, tid, a.par_out, a.cov_out, n, (size_t)i);
      o_chi2 = fc; o_score = fs;
      o_nh = __shfl_sync(gm, nh, src); o_nm = __shfl_sync(gm, nm, src); o_stat = 0;
      bt_step = t_last; bt_slot = fl2;
    } else if (bs_have) {
      o_chi2 = bs_chi2; o_score = bs_score; o_nh = bs_nh; o_nm = bs_nm; o_stat = bs_stat;
      bt_step = bs_step - 1; bt_slot = bs_parent; tail_step = bs_step; tail_val = bs_last;
    } else {                                                    // nothing qualifies: the seed itself, TRUNCATED
      o_chi2 = seed_chi2; o_nh = seed_nh; o_nm = 0; o_stat = seed_stat | ST_TRUNC; o_score = score_of(p, seed_nh, 0, seed_chi2);
      bt_step = seed_last; bt_slot = 0;
    }
    if (sub == 0) {
      a.chi2[i] = o_chi2; a.score[i] = o_score; a.nhits[i] = o_nh; a.nmiss[i] = o_nm; a.status[i] = o_stat;
    }
    // the winner's hit list: the 8 lanes bring the seed's trellis into shared memory (the propagated states are dead by
    // now), lane 0 walks it backwards, the 8 lanes write the plan steps
    const bool staged = (size_t)mpl * G * NS <= (size_t)NF * SL;
    unsigned* tsm = reinterpret_cast<unsigned*>(&sm.B[0][0]) + (size_t)sl * mpl * G;
    if (staged) {
      for (int s = 0; s <= max(bt_step, 0) && s < mpl; s++) tsm[s * G + sub] = trellis[(size_t)s * G + sub];
      __syncwarp(gm);
    }
    int slot = bt_slot;
    for (int s0 = ((mpl - 1) / G) * G; s0 >= 0; s0 -= G) {
      int mine = -2;
      if (sub == 0) {
        for (int s = min(s0 + G, mpl) - 1; s >= s0; s--) {
          int v = -2;
          int v2 = -2;
          if (s == tail_step) v = tail_val;
          else if (s <= bt_step) {
            const unsigned e = staged ? tsm[s * G + slot] : trellis[(size_t)s * G + slot];
            if (a.trellis2) v2 = a.trellis2[((size_t)i * mpl + s) * G + slot];
            v = (int)(e & 0x0fffffffu) - 2; slot = (int)(e >> 28);
          }
          sm.sel_t[(tid & ~(G - 1)) + (s - s0)] = v;
          sm.sel_hit2[(tid & ~(G - 1)) + (s - s0)] = v2;
        }
      }
      __syncwarp(gm);
      int mine2 = -2;
      if (s0 + sub < mpl) { mine = sm.sel_t[(tid & ~(G - 1)) + sub]; mine2 = sm.sel_hit2[(tid & ~(G - 1)) + sub]; }
      __syncwarp(gm);
      if (s0 + sub < mpl) { a.hit_ids[(size_t)(s0 + sub) * n + i] = mine; if (a.hit_ids2) a.hit_ids2[(size_t)(s0 + sub) * n + i] = mine2; }
    }
  }
  if (COUNT) {
    unsigned v[7] = {n_steps, n_pos, n_c2, n_acc, n_upd, n_rowt, n_rowo};
#pragma unroll
    for (int k = 0; k < 7; k++) {
      unsigned x = v[k];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
      if (lane == 0 && x) atomicAdd(&a.counters[k], (unsigned long long)x);
    }
  }
}

}  // namespace

namespace mkf {
// workspace of mkf_build_tracks: seed records, trellis, seed order, sort keys, bucket counts + scan partials
static size_t n_buckets_of(const mkf_ctx* c, int n_events) { return (size_t)n_events * c->g.n_plans * 256 + 1; }
size_t build_ws_bytes(const mkf_ctx* c, int n_events, int n_seeds) {
  const size_t n = (size_t)n_seeds, nbk = n_buckets_of(c, n_events);
  return align256(n * NW * 4) + align256(n * c->max_plan_len * G * 4) + 2 * align256(n * 4) + 2 * align256((nbk + 1) * 4) + scan_partial_bytes(nbk);
}
}  // namespace mkf

static int build_tracks_common(mkf_ctx* c, const mkf_hits* h, const mkf_hit_index* idx, const mkf_states* seeds,
                                const int* seed_event, const int* seed_hits, const signed char* plan, int max_plan_len,
                                mkf_states* out, float* chi2, float* score, int* nhits, int* nmiss, int* hit_ids, int* hit_ids2,
                                unsigned* status, void* ws, size_t ws_bytes, void* stream);

extern "C" int mkf_build_tracks(mkf_ctx* c, const mkf_hits* h, const mkf_hit_index* idx, const mkf_states* seeds,
                                const int* seed_event, const int* seed_hits, const signed char* plan, int max_plan_len,
                                mkf_states* out, float* chi2, float* score, int* nhits, int* nmiss, int* hit_ids,
                                unsigned* status, void* ws, size_t ws_bytes, void* stream) {
  return build_tracks_common(c, h, idx, seeds, seed_event, seed_hits, plan, max_plan_len, out, chi2, score, nhits, nmiss, hit_ids, nullptr,
                             status, ws, ws_bytes, stream);
}

extern "C" int mkf_build_tracks_overlap(mkf_ctx* c, const mkf_hits* h, const mkf_hit_index* idx, const mkf_states* seeds,
                                const int* seed_event, const int* seed_hits, const signed char* plan, int max_plan_len,
                                mkf_states* out, float* chi2, float* score, int* nhits, int* nmiss, int* hit_ids, int* hit_ids2,
                                unsigned* status, void* ws, size_t ws_bytes, void* stream) {
  if (!c) return MKF_INVALID_ARG;
  if (!h || !h->module || !hit_ids2) return fail(c, MKF_INVALID_ARG, "mkf_build_tracks_overlap: hits->module and hit_ids2 are needed");
  return build_tracks_common(c, h, idx, seeds, seed_event, seed_hits, plan, max_plan_len, out, chi2, score, nhits, nmiss, hit_ids, hit_ids2,
                             status, ws, ws_bytes, stream);
}

static int build_tracks_common(mkf_ctx* c, const mkf_hits* h, const mkf_hit_index* idx, const mkf_states* seeds,
                                const int* seed_event, const int* seed_hits, const signed char* plan, int max_plan_len,
                                mkf_states* out, float* chi2, float* score, int* nhits, int* nmiss, int* hit_ids, int* hit_ids2,
                                unsigned* status, void* ws, size_t ws_bytes, void* stream) {
  if (!c) return MKF_INVALID_ARG;
  if (!h || !idx || !seeds || !out) return fail(c, MKF_INVALID_ARG, "mkf_build_tracks: null argument");
  if (seeds->n < 0 || out->n != seeds->n || max_plan_len < 1) return fail(c, MKF_INVALID_ARG, "mkf_build_tracks: bad sizes");
  if (max_plan_len != c->max_plan_len) return fail(c, MKF_INVALID_ARG, "mkf_build_tracks: max_plan_len is not mkf_max_plan_len(ctx)");
  if (h->n_hits > (1 << 28) - 2) return fail(c, MKF_UNSUPPORTED, "mkf_build_tracks: n_hits > 2^28 - 2");
  if (seeds->n == 0) return MKF_OK;                      // nothing to do; array pointers may be null
  if (!seed_event || !seed_hits || !plan || !chi2 || !score || !nhits || !nmiss || !hit_ids || !status)
    return fail(c, MKF_INVALID_ARG, "mkf_build_tracks: null argument");
  if (!idx->bin_off || !idx->sorted_id || !idx->vmax || !h->layer_off || !h->x || !h->y || !h->z || !h->V ||
      !seeds->par || !seeds->cov || !seeds->q || !out->par || !out->cov)
    return fail(c, MKF_INVALID_ARG, "mkf_build_tracks: null array");
  if (h->n_events < 1) return fail(c, MKF_INVALID_ARG, "mkf_build_tracks: no events");
  if (c->g.n_phi > 255 || c->g.n_eta > 255) return fail(c, MKF_UNSUPPORTED, "mkf_build_tracks: more than 255 phi or eta bins");
  const size_t tr2_bytes = hit_ids2 ? align256((size_t)seeds->n * max_plan_len * G * 4) : 0;
  const size_t need = build_ws_bytes(c, h->n_events, seeds->n) + tr2_bytes;
  if (ws_bytes < need || !ws) return fail(c, MKF_WORKSPACE_TOO_SMALL, "mkf_build_tracks: workspace too small");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t n = (size_t)seeds->n, nbk = n_buckets_of(c, h->n_events);
  char* w = (char*)ws;
  BuildArgs a;
  a.hits = hits_dev(h);
  a.bin_off = idx->bin_off; a.sorted_id = idx->sorted_id; a.vmax = idx->vmax; a.packed = (const float4*)idx->packed;
  a.n = seeds->n; a.par = seeds->par; a.cov = seeds->cov; a.q = seeds->q; a.seed_event = seed_event; a.seed_hits = seed_hits;
  a.plan = plan; a.max_plan_len = max_plan_len;
  a.par_out = out->par; a.cov_out = out->cov; a.chi2 = chi2; a.score = score; a.nhits = nhits; a.nmiss = nmiss;
  a.hit_ids = hit_ids; a.status = status;
  a.wseed = (float*)w; w += align256(n * NW * 4);
  a.trellis = (unsigned*)w; w += align256(n * max_plan_len * G * 4);
  int* order = (int*)w; w += align256(n * 4);
  a.order = order;
  a.key = (unsigned*)w; w += align256(n * 4);
  a.bucket = (unsigned*)w; w += align256((nbk + 1) * 4);
  unsigned* bucket_off = (unsigned*)w; w += align256((nbk + 1) * 4);
  unsigned* partial = (unsigned*)w; w += scan_partial_bytes(nbk);
  a.trellis2 = hit_ids2 ? (int*)w : nullptr;
  a.hit_ids2 = hit_ids2;
  a.n_buckets = (int)nbk;
  a.counters = c->build_counters;
  cudaError_t e = cudaMemsetAsync(a.bucket, 0, nbk * 4, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "mkf_build_tracks: memset");
  bs_seed_kernel<<<(a.n + 127) / 128, 128, 0, st>>>(c->g, c->p, a);
  MKF_LAUNCHED(c, "bs_seed_kernel");
  { const int rc = exclusive_scan_u32(c, a.bucket, nbk, partial, bucket_off, (unsigned)a.n, st); if (rc) return rc; }
  bs_order_kernel<<<(a.n + 255) / 256, 256, 0, st>>>(a.n, a.key, a.bucket, order);
  MKF_LAUNCHED(c, "bs_order_kernel");
  const size_t smem = sizeof(Smem);
  const int grid = (a.n + NS - 1) / NS;
  // four instances: with / without the work counters, hits from the packed index / gathered by id
  void (*kern)(GeomDev, ParamsDev, BuildArgs) =
      a.counters ? (a.packed ? mkf_build_kernel<true, true> : mkf_build_kernel<true, false>)
                 : (a.packed ? mkf_build_kernel<false, true> : mkf_build_kernel<false, false>);
  e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return cuda_fail(c, e, "mkf_build_tracks: shared memory attribute");
  kern<<<grid, BT, smem, st>>>(c->g, c->p, a);
  MKF_LAUNCHED(c, "mkf_build_kernel");
  return MKF_OK;
}
