// mkf_build.cu — a12 / C9: combinatorial track building ("combinatorial search ... from a seed in the
// innermost layers, proceeding outwards", "only the best ranking ones are cloned at each layer (with
// a per-seed cap)", PAPER.md:5 short-track preservation).
//
// Mapping: 8 lanes of a warp own one seed (4 seeds per warp); lane k holds live candidate k (rank order) with its
// state and covariance in registers. Per layer: every live lane propagates its candidate (a2-a4), scans the
// phi/eta bins of its window (a5) reading the packed hit records (16-byte positions first: most are rejected before
// their covariance is read), keeps its own best MAX_CAND hits by chi2 in a sorted list in shared memory (a6); the group then picks the top max_cand children of the whole seed
// with 8-lane shuffle tournaments under the total order U14 (a8), the winners fetch their parent's state with
// shuffles and update it (a7). The hit lists are a trellis in shared memory (per step and slot: hit id and
// parent slot), so cloning a candidate costs one 4-byte entry; the winner's list is read back at the end.
// Stopped candidates are offered to the seed's `best short` slot (a9), whose state lives in the output arrays.
#include "mkf_ctx.h"

using namespace mkf;

namespace {

constexpr int G = 8;                 // lanes per seed == MAX_CAND
#ifndef MKF_BUILD_BLOCK
#define MKF_BUILD_BLOCK 64
#endif
constexpr int BUILD_BLOCK = MKF_BUILD_BLOCK;     // 8 seeds per CTA (64 threads: 2193 events/s on configs[4]; 128: 2108, 32: 2178)
constexpr int HIT_NONE = 0x7fffffff; // "hit id" of miss / pass-through children in the order U14
static_assert(G == MAX_CAND, "one lane per candidate slot");

struct BuildArgs {
  HitsDev hits;
  const unsigned* bin_off; const int* sorted_id; const float* vmax; const float4* packed;
  int n; const float* par; const float* cov; const signed char* q; const int* seed_event; const int* seed_hits;
  const signed char* plan; int max_plan_len;
  float* par_out; float* cov_out; float* chi2; float* score; int* nhits; int* nmiss; int* hit_ids; unsigned* status;
};

__device__ __forceinline__ float score_of(const ParamsDev& p, int nh, int nm, float chi2) {
  return p.score_hit * (float)nh - p.score_miss * (float)nm - chi2;
}

// U14: does child a rank before child b?
__device__ __forceinline__ bool before(float sa, float ca, int pa, int ha, float sb, float cb, int pb, int hb) {
  if (sa != sb) return sa > sb;
  if (ca != cb) return ca < cb;
  if (pa != pb) return pa < pb;
  return ha < hb;
}

__device__ __forceinline__ void load_packed(Hit& H, int& id, const float4 a, const float4* __restrict__ cov) {
  const float4 b = __ldg(cov), c = __ldg(cov + 1);
  H.x = a.x; H.y = a.y; H.z = a.z; id = __float_as_int(a.w);
  H.v[0] = b.x; H.v[1] = b.y; H.v[2] = b.z; H.v[3] = b.w; H.v[4] = c.x; H.v[5] = c.y;
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

#define SHFL_STATE(S, src, gm)                                           \
  do {                                                                   \
    S.x = __shfl_sync(gm, S.x, src); S.y = __shfl_sync(gm, S.y, src); S.z = __shfl_sync(gm, S.z, src);       \
    S.xl = __shfl_sync(gm, S.xl, src); S.yl = __shfl_sync(gm, S.yl, src); S.zl = __shfl_sync(gm, S.zl, src); \
    S.ipt = __shfl_sync(gm, S.ipt, src); S.phi = __shfl_sync(gm, S.phi, src); S.th = __shfl_sync(gm, S.th, src); \
    S.cph = __shfl_sync(gm, S.cph, src); S.sph = __shfl_sync(gm, S.sph, src);                                 \
    S.cth = __shfl_sync(gm, S.cth, src); S.sth = __shfl_sync(gm, S.sth, src);                                 \
    S.f.kind = __shfl_sync(gm, S.f.kind, src); S.f.cb = __shfl_sync(gm, S.f.cb, src); S.f.sb = __shfl_sync(gm, S.f.sb, src); \
    _Pragma("unroll") for (int k_ = 0; k_ < 10; k_++) S.u[k_] = __shfl_sync(gm, S.u[k_], src);             \
    _Pragma("unroll") for (int k_ = 0; k_ < 5; k_++) S.d[k_] = __shfl_sync(gm, S.d[k_], src);              \
  } while (0)

#ifndef MKF_BUILD_MIN_BLOCKS
#define MKF_BUILD_MIN_BLOCKS 16
#endif
__global__ void __launch_bounds__(BUILD_BLOCK, MKF_BUILD_MIN_BLOCKS) mkf_build_kernel(const __grid_constant__ GeomDev g,
                                                                const __grid_constant__ ParamsDev p,
                                                                const __grid_constant__ BuildArgs a) {
  extern __shared__ unsigned trellis_all[];                  // [seed in CTA][step][slot]
  const int lane = threadIdx.x & 31;
  const int sub = lane & (G - 1);                            // candidate slot
  const int gbase = lane & ~(G - 1);
  const unsigned gm = 0xffu << gbase;
  const int seed_in_cta = threadIdx.x / G;
  const int i = blockIdx.x * (BUILD_BLOCK / G) + seed_in_cta;
  const bool have_seed = i < a.n;
  const size_t n = (size_t)a.n;
  const int mpl = a.max_plan_len;
  unsigned* trellis = trellis_all + (size_t)seed_in_cta * mpl * G;
  // per-thread list of accepted hits of the current layer, [k][thread] (bank-conflict free): chi2, hit id
  float* hc2 = reinterpret_cast<float*>(trellis_all + (size_t)(BUILD_BLOCK / G) * mpl * G) + threadIdx.x;
  int* hid = reinterpret_cast<int*>(hc2 - threadIdx.x + G * BUILD_BLOCK) + threadIdx.x;
  const int nb = g.n_phi * g.n_eta;

  // ---- seed phase: slot 0 fits the seed through its own three hits (U18b) --------------------------------
  KState S;
  float chi2 = 0.f; int nh = 0, nm = 0, consec = 0; unsigned stat = 0;
  bool live = false;
  int p0 = 0, plen = 0, ev = 0, last_step = -1;
  float aq = 0.f;
  bool seed_ok = false;
  if (have_seed) {
    const int pl = a.plan[i];
    p0 = g.plan_off[pl];
    plen = min(g.plan_off[pl + 1] - p0, mpl);
    ev = a.seed_event[i];
    aq = -(float)a.q[i] * KAPPA * g.bz;
    for (int s = sub; s < mpl; s += G) trellis[s * G + 0] = 0u;          // hit code 0 == -2 (not crossed), parent 0
  }
  __syncwarp(gm);
  if (have_seed && sub == 0) {
    load_params(S, a.par, n, (size_t)i);
    bool has_ud = false;
    const int* loff = a.hits.layer_off + (size_t)ev * (g.n_layers + 1);
    seed_ok = true;
    for (int k = 0; k < 3 && seed_ok; k++) {
      const int hid = a.seed_hits[(size_t)k * n + i];
      int lay = -1;
      for (int l = 0; l < g.n_layers; l++) if (hid >= loff[l] && hid < loff[l + 1]) { lay = l; break; }
      int step = -1;
      for (int s = last_step + 1; s < plen; s++) if ((int)g.plan_layers[p0 + s] == lay) { step = s; break; }
      if (step < 0) { stat |= ST_TRUNC; seed_ok = false; break; }
      const LayerDev L = g.layers[lay];
      const unsigned rc = step_to_layer(S, !has_ud, a.cov, n, (size_t)i, L, aq, p.graze_cos_min, p.material_flags, false);
      if (rc) { stat |= rc; seed_ok = false; break; }
      has_ud = true;
      Hit H; load_hit(H, a.hits, hid);
      SInv o; float c2;
      hit_to_local(S, H, o);
      if (!kalman_update(S, o, c2)) { stat |= ST_S_NOT_PD; seed_ok = false; break; }
      chi2 += c2; nh++; last_step = step;
      trellis[step * G + 0] = (unsigned)(hid + 2);
    }
    // fallback output: the seed candidate itself (C9 last line); overwritten by best_short / the final winner
    if (has_ud) store_state(S, a.par_out, a.cov_out, n, (size_t)i);
    else copy_seed(a.par, a.cov, a.par_out, a.cov_out, n, (size_t)i);
    live = seed_ok;
  }
  seed_ok = __shfl_sync(gm, (int)seed_ok, gbase) != 0;
  last_step = __shfl_sync(gm, last_step, gbase);
  const float seed_chi2 = __shfl_sync(gm, chi2, gbase);
  const int seed_nh = __shfl_sync(gm, nh, gbase);
  const unsigned seed_stat = __shfl_sync(gm, stat, gbase);

  // best short candidate of the seed (replicated in every lane of the group)
  bool bs_have = false; float bs_score = 0.f, bs_chi2 = 0.f; int bs_nh = 0, bs_nm = 0, bs_step = 0, bs_parent = 0, bs_last = -2;
  unsigned bs_stat = 0;
  int t_last = last_step;                                    // last step at which the live set was rewritten
  int n_live = seed_ok ? 1 : 0;

  for (int s = 0; s < mpl; s++) {
    const bool active = have_seed && seed_ok && s > last_step && s < plen && n_live > 0;   // uniform in the group
    if (!active) continue;
    const int lay = g.plan_layers[p0 + s];
    const LayerDev L = g.layers[lay];
    const size_t seg = (size_t)ev * g.n_layers + lay;

    // ---- each live lane: propagate, scan its window, keep its own best hits ------------------------------
    int n_hitc = 0, head = 0;             // accepted hits in hc2/hid (sorted), next one to offer
    bool miss_avail = false, pass_avail = false;
    bool offer = false; int offer_phase = 0; float offer_score = 0.f; int offer_nm = 0;
    if (live) {
      const unsigned rc = step_to_layer(S, false, a.cov, n, (size_t)i, L, aq, p.graze_cos_min, p.material_flags, true);
      if (rc & (ST_UNREACH | ST_SKIP_ACC)) {
        pass_avail = true;                                   // silent skip: competes unchanged (C9.1)
      } else if (rc) {                                       // grazing / energy exhausted: the candidate stops
        stat |= rc;
        if (nh >= p.min_hits_keep) { offer = true; offer_phase = 0; offer_nm = nm; offer_score = score_of(p, nh, nm, chi2); }
      } else {
        float tt, tz, zz;
        cov_aa(S, tt, tz, zz);
        int e0, e1, w0, wn;
        window(g, L, p.chi2_cut, S, tt, zz, a.vmax[2 * seg], a.vmax[2 * seg + 1], e0, e1, w0, wn);
        const float lim1 = p.chi2_cut * (tt + a.vmax[2 * seg]) * 1.0001f;
        const float lim2 = p.chi2_cut * (zz + (L.kind == 0 ? a.vmax[2 * seg + 1] : a.vmax[2 * seg])) * 1.0001f;
        const unsigned* boff = a.bin_off + seg * (size_t)nb;
        for (int ie = e0; ie <= e1; ie++) {
          const unsigned* row = boff + ie * g.n_phi;
#pragma unroll 1
          for (int part = 0; part < 2; part++) {
            unsigned tb, te;
            if (part == 0) { tb = row[w0]; te = row[min(w0 + wn, g.n_phi)]; }
            else { if (w0 + wn <= g.n_phi) break; tb = row[0]; te = row[w0 + wn - g.n_phi]; }
            float4 qn = make_float4(0.f, 0.f, 0.f, 0.f);
            if (a.packed && tb < te) qn = __ldg(a.packed + tb);
            for (unsigned t = tb; t < te; t++) {
              Hit H; int id;
              if (a.packed) {
                // position first: chi2 >= (e.r)^2 / (e^T S e) for the unit vectors e = w1, w2 (Cauchy-Schwarz, U11),
                // so most hits of the padded bins are rejected before their covariance is read; the next record's
                // position is already in flight
                const float4 q0 = qn;
                if (t + 1 < te) qn = __ldg(a.packed + t + 1);
                const float rx = (q0.x - S.x) - S.xl, ry = (q0.y - S.y) - S.yl, rz = (q0.z - S.z) - S.zl;
                const float r1 = S.f.kind == 0 ? S.f.cb * ry - S.f.sb * rx : rx, r2 = S.f.kind == 0 ? rz : ry;
                if (r1 * r1 > lim1 || r2 * r2 > lim2) continue;
                load_packed(H, id, q0, a.packed + (size_t)a.hits.n_hits + (size_t)2 * t);
              } else { id = a.sorted_id[t]; load_hit(H, a.hits, id); }
              SInv o; float c2;
              if (!chi2_local(S, tt, tz, zz, H, o, c2)) continue;
              if (c2 < p.chi2_cut) {
                // kept sorted by (chi2, id) in shared memory: lists are short (1-2 entries on average), so the
                // insertion is a handful of divergent instructions and no register array is needed
                int k = n_hitc;
                if (n_hitc == G) {
                  const float wv = hc2[(G - 1) * BUILD_BLOCK]; const int wi = hid[(G - 1) * BUILD_BLOCK];
                  k = (c2 < wv || (c2 == wv && id < wi)) ? G - 1 : -1;
                } else n_hitc++;
                if (k >= 0) {
                  while (k > 0) {
                    const float pv = hc2[(k - 1) * BUILD_BLOCK]; const int pi = hid[(k - 1) * BUILD_BLOCK];
                    if (!(c2 < pv || (c2 == pv && id < pi))) break;
                    hc2[k * BUILD_BLOCK] = pv; hid[k * BUILD_BLOCK] = pi; k--;
                  }
                  hc2[k * BUILD_BLOCK] = c2; hid[k * BUILD_BLOCK] = id;
                }
              }
            }
          }
        }
        // miss child (C9.5): stopped if it reaches the consecutive-miss limit
        if (consec + 1 >= p.max_consec_miss) {
          if (nh >= p.min_hits_keep) { offer = true; offer_phase = 1; offer_nm = nm + 1; offer_score = score_of(p, nh, nm + 1, chi2); }
        } else miss_avail = true;
      }
    }

    // ---- offers to best_short (C9.6): best offer of this layer, then strict comparison with the holder ------
    {
      float os = offer ? offer_score : -INFINITY, oc = chi2; int ok = offer_phase * G + sub;
      int ol = sub;
#pragma unroll
      for (int d = 1; d < G; d <<= 1) {
        const float s2 = __shfl_xor_sync(gm, os, d), c2 = __shfl_xor_sync(gm, oc, d);
        const int k2 = __shfl_xor_sync(gm, ok, d), l2 = __shfl_xor_sync(gm, ol, d);
        const bool take = (s2 != os) ? (s2 > os) : ((c2 != oc) ? (c2 < oc) : (k2 < ok));
        if (take) { os = s2; oc = c2; ok = k2; ol = l2; }
      }
      if (os > -INFINITY && (!bs_have || os > bs_score || (os == bs_score && oc < bs_chi2))) {
        const int src = gbase + ol;
        if (sub == ol) store_state(S, a.par_out, a.cov_out, n, (size_t)i);
        bs_have = true; bs_score = os; bs_chi2 = oc;
        bs_nh = __shfl_sync(gm, nh, src); bs_nm = __shfl_sync(gm, offer_nm, src);
        bs_stat = __shfl_sync(gm, stat, src);
        bs_step = s; bs_parent = ol; bs_last = (ok >= G) ? -1 : -2;
      }
    }

    // ---- top max_cand children of the seed (U14) --------------------------------------------------------
    const float base_hit = score_of(p, nh + 1, nm, chi2);     // hit child: base_hit - c2_hit
    const float sc_miss = score_of(p, nh, nm + 1, chi2), sc_pass = score_of(p, nh, nm, chi2);
    int my_parent = sub, my_hit = -2, my_kind = -1;           // what this slot becomes
    int n_new = 0;
    for (int r = 0; r < p.max_cand; r++) {
      float hs, hc; int hh, hk;                               // head child of this lane
      if (head < n_hitc) { const float c2h = hc2[head * BUILD_BLOCK]; hs = base_hit - c2h; hc = chi2 + c2h; hh = hid[head * BUILD_BLOCK]; hk = 0; }
      else if (miss_avail) { hs = sc_miss; hc = chi2; hh = HIT_NONE; hk = 1; }
      else if (pass_avail) { hs = sc_pass; hc = chi2; hh = HIT_NONE; hk = 2; }
      else { hs = -INFINITY; hc = INFINITY; hh = HIT_NONE; hk = 3; }
      float ws = hs, wc = hc; int wp = sub, wh = hh, wk = hk;
#pragma unroll
      for (int d = 1; d < G; d <<= 1) {
        const float s2 = __shfl_xor_sync(gm, ws, d), c2 = __shfl_xor_sync(gm, wc, d);
        const int p2 = __shfl_xor_sync(gm, wp, d), h2 = __shfl_xor_sync(gm, wh, d), k2 = __shfl_xor_sync(gm, wk, d);
        if (before(s2, c2, p2, h2, ws, wc, wp, wh)) { ws = s2; wc = c2; wp = p2; wh = h2; wk = k2; }
      }
      if (!(ws > -INFINITY)) break;                           // pool exhausted (uniform in the group)
      if (sub == wp) {                                        // the winner lane pops its head
        if (wk == 0) {
          head++;
        } else if (wk == 1) miss_avail = false;
        else pass_avail = false;
      }
      if (sub == r) { my_parent = wp; my_kind = wk; my_hit = wk == 0 ? wh : (wk == 1 ? -1 : -2); }
      n_new = r + 1;
    }

    // ---- the new live set: fetch the parent's state, update with the hit -----------------------------------
    {
      const int src = gbase + my_parent;
      SHFL_STATE(S, src, gm);
      chi2 = __shfl_sync(gm, chi2, src);
      nh = __shfl_sync(gm, nh, src); nm = __shfl_sync(gm, nm, src); consec = __shfl_sync(gm, consec, src);
      stat = __shfl_sync(gm, stat, src);
    }
    live = sub < n_new;
    if (live) {
      if (my_kind == 1) { nm++; consec++; }
      else if (my_kind == 0) {
        Hit H; load_hit(H, a.hits, my_hit);
        SInv o; float c2;
        hit_to_local(S, H, o);
        if (kalman_update(S, o, c2)) {
          chi2 += c2; nh++; consec = 0;
          if (!state_finite(S)) live = false;                 // dropped (C9: NaN child)
        } else live = false;
      }
    }
    // keep the live lanes contiguous in rank order (only needed after a dropped child)
    const unsigned alive = (__ballot_sync(gm, live) >> gbase) & 0xffu;
    if (alive != ((1u << n_new) - 1u)) {
      const int cnt = __popc(alive);
      const int pick = sub < cnt ? (int)__fns(alive, 0, sub + 1) : sub;
      const int src = gbase + pick;
      SHFL_STATE(S, src, gm);
      chi2 = __shfl_sync(gm, chi2, src);
      nh = __shfl_sync(gm, nh, src); nm = __shfl_sync(gm, nm, src); consec = __shfl_sync(gm, consec, src);
      stat = __shfl_sync(gm, stat, src);
      my_parent = __shfl_sync(gm, my_parent, src); my_hit = __shfl_sync(gm, my_hit, src);
      n_new = cnt; live = sub < cnt;
    }
    if (live) trellis[s * G + sub] = (unsigned)(my_hit + 2) | ((unsigned)my_parent << 28);
    n_live = n_new;
    t_last = s;
    __syncwarp(gm);
  }

  if (!have_seed) return;
  // ---- final choice: best of live U {best_short} (C9) -------------------------------------------------------
  float fs = (live && nh >= p.min_hits_keep) ? score_of(p, nh, nm, chi2) : -INFINITY, fc = chi2; int fl = sub;
#pragma unroll
  for (int d = 1; d < G; d <<= 1) {
    const float s2 = __shfl_xor_sync(gm, fs, d), c2 = __shfl_xor_sync(gm, fc, d);
    const int l2 = __shfl_xor_sync(gm, fl, d);
    const bool take = (s2 != fs) ? (s2 > fs) : ((c2 != fc) ? (c2 < fc) : (l2 < fl));
    if (take) { fs = s2; fc = c2; fl = l2; }
  }
  const bool live_wins = fs > -INFINITY && !(bs_have && (bs_score > fs || (bs_score == fs && bs_chi2 < fc)));
  float o_chi2, o_score; int o_nh, o_nm, bt_step, bt_slot, tail_step = -1, tail_val = -2; unsigned o_stat;
  if (live_wins) {
    const int src = gbase + fl;
    if (sub == fl) store_state(S, a.par_out, a.cov_out, n, (size_t)i);
    o_chi2 = fc; o_score = fs;
    o_nh = __shfl_sync(gm, nh, src); o_nm = __shfl_sync(gm, nm, src); o_stat = __shfl_sync(gm, stat, src);
    bt_step = t_last; bt_slot = fl;
  } else if (bs_have) {
    o_chi2 = bs_chi2; o_score = bs_score; o_nh = bs_nh; o_nm = bs_nm; o_stat = bs_stat;
    bt_step = bs_step - 1; bt_slot = bs_parent; tail_step = bs_step; tail_val = bs_last;
  } else {                                                    // nothing qualifies: the seed itself, TRUNCATED
    o_chi2 = seed_chi2; o_nh = seed_nh; o_nm = 0; o_stat = seed_stat | ST_TRUNC; o_score = score_of(p, seed_nh, 0, seed_chi2);
    bt_step = last_step; bt_slot = 0;
  }
  __syncwarp(gm);
  if (sub == 0) {
    a.chi2[i] = o_chi2; a.score[i] = o_score; a.nhits[i] = o_nh; a.nmiss[i] = o_nm; a.status[i] = o_stat;
    int slot = bt_slot;
    for (int s = mpl - 1; s >= 0; s--) {
      int v = -2;
      if (s == tail_step) v = tail_val;
      else if (s <= bt_step) { const unsigned e = trellis[s * G + slot]; v = (int)(e & 0x0fffffffu) - 2; slot = (int)(e >> 28); }
      a.hit_ids[(size_t)s * n + i] = v;
    }
  }
}

}  // namespace

namespace mkf {
size_t build_smem_bytes(int max_plan_len) {
  return (size_t)(BUILD_BLOCK / G) * max_plan_len * G * sizeof(unsigned) + (size_t)2 * G * BUILD_BLOCK * sizeof(float);
}
}

extern "C" int mkf_build_tracks(mkf_ctx* c, const mkf_hits* h, const mkf_hit_index* idx, const mkf_states* seeds,
                                const int* seed_event, const int* seed_hits, const signed char* plan, int max_plan_len,
                                mkf_states* out, float* chi2, float* score, int* nhits, int* nmiss, int* hit_ids,
                                unsigned* status, void* ws, size_t ws_bytes, void* stream) {
  (void)ws; (void)ws_bytes;
  if (!c) return MKF_INVALID_ARG;
  if (!h || !idx || !seeds || !out) return fail(c, MKF_INVALID_ARG, "mkf_build_tracks: null argument");
  if (seeds->n < 0 || out->n != seeds->n || max_plan_len < 1) return fail(c, MKF_INVALID_ARG, "mkf_build_tracks: bad sizes");
  if (h->n_hits >= (1 << 28)) return fail(c, MKF_UNSUPPORTED, "mkf_build_tracks: n_hits >= 2^28");
  if (seeds->n == 0) return MKF_OK;                      // nothing to do; array pointers may be null
  if (!seed_event || !seed_hits || !plan || !chi2 || !score || !nhits || !nmiss || !hit_ids || !status)
    return fail(c, MKF_INVALID_ARG, "mkf_build_tracks: null argument");
  if (!idx->bin_off || !idx->sorted_id || !idx->vmax || !h->layer_off || !h->x || !h->y || !h->z || !h->V ||
      !seeds->par || !seeds->cov || !seeds->q || !out->par || !out->cov)
    return fail(c, MKF_INVALID_ARG, "mkf_build_tracks: null array");
  const size_t smem = build_smem_bytes(max_plan_len);
  if (smem > 200 * 1024) return fail(c, MKF_UNSUPPORTED, "mkf_build_tracks: plan too long for the shared-memory trellis");
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(mkf_build_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cuda_fail(c, e, "mkf_build_tracks: shared memory attribute");
  }
  BuildArgs a;
  a.hits = hits_dev(h);
  a.bin_off = idx->bin_off; a.sorted_id = idx->sorted_id; a.vmax = idx->vmax; a.packed = (const float4*)idx->packed;
  a.n = seeds->n; a.par = seeds->par; a.cov = seeds->cov; a.q = seeds->q; a.seed_event = seed_event; a.seed_hits = seed_hits;
  a.plan = plan; a.max_plan_len = max_plan_len;
  a.par_out = out->par; a.cov_out = out->cov; a.chi2 = chi2; a.score = score; a.nhits = nhits; a.nmiss = nmiss;
  a.hit_ids = hit_ids; a.status = status;
  const int seeds_per_cta = BUILD_BLOCK / G;
  const int grid = (a.n + seeds_per_cta - 1) / seeds_per_cta;
  mkf_build_kernel<<<grid, BUILD_BLOCK, smem, (cudaStream_t)stream>>>(c->g, c->p, a);
  MKF_LAUNCHED(c, "mkf_build_kernel");
  return MKF_OK;
}
