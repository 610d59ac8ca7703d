// mkf_dev.cuh — device-side tables passed by value as kernel parameters, and SoA load/store helpers.
#pragma once
#include "kf_math.cuh"

namespace mkf {

constexpr int MAX_LAYERS = 64, MAX_PLANS = 8, MAX_PLAN_STEPS = 192, MAX_CAND = 8;

// Geometry + parameters: ~2.1 KB, lives in the kernel parameter (constant) bank.
struct GeomDev {
  int n_layers, n_plans, n_phi, n_eta;
  float bz;
  int plan_off[MAX_PLANS + 1];
  unsigned char plan_layers[MAX_PLAN_STEPS];
  LayerDev layers[MAX_LAYERS];
  float bz_layer[MAX_LAYERS];          // R13: field of the step that ends on the layer (all = bz without the hook)
};

struct ParamsDev {
  float chi2_cut; int max_cand, max_consec_miss, min_hits_keep;
  float score_hit, score_miss, graze_cos_min; int material_flags; float dup_frac;
};

struct HitsDev { int n_events, n_hits; const int* layer_off; const float *x, *y, *z, *V; const float4* rec; const int* module; };

// Parameters of a caller's state; the covariance is read separately by the first propagation (commit_first).
MKF_HD void load_params(KState& S, const float* par, size_t n, size_t i) {
  S.x = par[i]; S.y = par[n + i]; S.z = par[2 * n + i];
  S.xl = 0.f; S.yl = 0.f; S.zl = 0.f;
  S.ipt = par[3 * n + i]; S.phi = par[4 * n + i]; S.th = par[5 * n + i];
  sincos_f(S.phi, &S.sph, &S.cph);
  sincos_f(S.th, &S.sth, &S.cth);
  S.f.kind = 0; S.f.cb = 1.f; S.f.sb = 0.f;
#pragma unroll
  for (int k = 0; k < 10; k++) S.u[k] = 0.f;
#pragma unroll
  for (int k = 0; k < 5; k++) S.d[k] = 0.f;
}

MKF_HD void load_cov(float* c, const float* cov, size_t n, size_t i) {
#pragma unroll
  for (int k = 0; k < 21; k++) c[k] = cov[(size_t)k * n + i];
}

// State with factors -> the caller's layout (global packed 6x6).
MKF_HD void store_state(const KState& S, float* par, float* cov, size_t n, size_t i) {
  par[i] = S.x + S.xl; par[n + i] = S.y + S.yl; par[2 * n + i] = S.z + S.zl;
  par[3 * n + i] = S.ipt; par[4 * n + i] = wrap_phi(S.phi); par[5 * n + i] = S.th;
  float l[15], c[21];
  ud_to_cov(S.u, S.d, l);
  cov_from_local(l, S.f, c);
#pragma unroll
  for (int k = 0; k < 21; k++) cov[(size_t)k * n + i] = c[k];
}

// A state that never completed a propagation: the caller's seed goes out as it came in.
MKF_HD void copy_seed(const float* par, const float* cov, float* par_out, float* cov_out, size_t n, size_t i) {
#pragma unroll
  for (int k = 0; k < 6; k++) par_out[(size_t)k * n + i] = par[(size_t)k * n + i];
#pragma unroll
  for (int k = 0; k < 21; k++) cov_out[(size_t)k * n + i] = cov[(size_t)k * n + i];
}

// One filter step up to (not including) the update. `first`: the state has no factors yet (they are made from the
// caller's covariance). Returns 0 and the advanced state, or a status bit with the state unchanged.
MKF_HD unsigned step_to_layer(KState& S, bool first, const float* cov, size_t n, size_t i, const LayerDev& L, float aq,
                              float graze_cos_min, int mflags, bool check_acc) {
  Prop P;
  const unsigned rc = propagate_geom(S, L, aq, graze_cos_min, mflags, check_acc, P);
  if (rc) return rc;
  if (first) { float c[21]; load_cov(c, cov, n, i); commit_first(S, c, P, mflags); }
  else commit_step(S, P, mflags);
  return 0;
}

// packed hit index (mkf_hit_index.packed): first float4 of the covariance block; even, so that every 32-byte covariance
// record is one whole sector
MKF_HD size_t packed_cov_off(int n_hits) { return (size_t)n_hits + (size_t)(n_hits & 1); }

MKF_HD void load_hit(Hit& H, const HitsDev& h, int id);
// PLANES: the hits are known to come as SoA planes (no test of the record pointer per hit); otherwise load_hit decides.
// (An instance with the records known at compile time was measured too: 22.4 against 23.5 G layer-steps/s.)
template <bool PLANES>
MKF_HD void load_hit_t(Hit& H, const HitsDev& h, int id) {
  if (PLANES) {
    const size_t nh = (size_t)h.n_hits;
    H.x = h.x[id]; H.y = h.y[id]; H.z = h.z[id];
#pragma unroll
    for (int k = 0; k < 6; k++) H.v[k] = h.V[(size_t)k * nh + id];
  } else load_hit(H, h, id);
}

MKF_HD void load_hit(Hit& H, const HitsDev& h, int id) {
#ifdef __CUDA_ARCH__
  if (h.rec) {                                                   // 48-byte record: 2 sectors instead of 9 for a scattered id
    const float4* r = h.rec + (size_t)3 * id;
    const float4 a = __ldg(r), b = __ldg(r + 1), c = __ldg(r + 2);
    H.x = a.x; H.y = a.y; H.z = a.z; H.v[0] = a.w; H.v[1] = b.x; H.v[2] = b.y; H.v[3] = b.z; H.v[4] = b.w; H.v[5] = c.x;
    return;
  }
#endif
  const size_t nh = (size_t)h.n_hits;
  H.x = h.x[id]; H.y = h.y[id]; H.z = h.z[id];
#pragma unroll
  for (int k = 0; k < 6; k++) H.v[k] = h.V[(size_t)k * nh + id];
}

// ---- fit of one track (C7) ------------------------------------------------------------------------------
struct FitArgs {
  HitsDev hits;
  int n;                       // tracks of this launch
  int ld;                      // plane stride of every per-track array (>= n; the host entry points launch on track ranges)
  const float* par; const float* cov; const signed char* q; const signed char* plan;
  const int* track_hits; int max_plan_len;
  float* par_out; float* cov_out; float* chi2; int* nfit; unsigned* status;
};

// The track keeps its last good state when a step fails. Failures found before the covariance is touched
// (unreachable, grazing, energy exhausted) leave the state as it was; the two that can only be seen after the
// update (S not positive definite, non-finite result) re-run the track from its seed up to the failing step.
// STRAG: the context asks for energy-loss straggling (material flag 4, R12); without it that code is not compiled in.
template <bool STRAG, bool PLANES>
MKF_HD void fit_one(const GeomDev& g, const ParamsDev& p, const FitArgs& a, int i) {
  const int mflags = STRAG ? p.material_flags : (p.material_flags & 3);
  const size_t n = (size_t)a.ld;
  const int pl = a.plan[i];
  if ((unsigned)pl >= (unsigned)g.n_plans) {                     // not a plan of this geometry: the seed goes out, flagged
    copy_seed(a.par, a.cov, a.par_out, a.cov_out, n, (size_t)i);
    a.chi2[i] = 0.f; a.nfit[i] = 0; a.status[i] = ST_TRUNC;
    return;
  }
  const int p0 = g.plan_off[pl];
  int plen = g.plan_off[pl + 1] - p0;
  if (plen > a.max_plan_len) plen = a.max_plan_len;
  const float qk = -(float)a.q[i] * KAPPA;                       // a = qk Bz of the step (R13)
  unsigned stat = 0;
  int stop_at = plen;
#ifdef __CUDA_ARCH__
  const unsigned wmask = __activemask();                         // the threads of this warp that own a track
#endif
  KState S;
  float c2tot; int nf;
  // pass 0 runs without per-step finiteness checks; only if its result is not finite, pass 1 finds the step
  // and pass 2 stops before it
  for (int pass = 0; pass < 3; pass++) {
    const bool check = pass == 1;
    load_params(S, a.par, n, (size_t)i);
    c2tot = 0.f; nf = 0;
    bool redo = false, stopped = false;
    const int* th = a.track_hits + i;
    const int stop_at_loop = stop_at;
    int hid_next = stop_at > 0 ? *th : -1;                       // the hit id is fetched one step ahead
    // every thread of the warp goes through every iteration and the warp is re-joined at its top: a thread that
    // skipped a layer without a hit (or stopped) would otherwise run ahead of its warp and never rejoin it
    // (measured on hit lists with 5 % gaps: 14.7 instead of 34.5 G layer-steps/s)
    for (int s = 0; s < stop_at_loop; s++) {
#ifdef __CUDA_ARCH__
      __syncwarp(wmask);
#endif
      const int hid = hid_next;
      th += n;
      hid_next = s + 1 < stop_at_loop ? *th : -1;
      if (hid < 0 || stopped) continue;
      if (hid >= a.hits.n_hits) { stat |= ST_TRUNC; stopped = true; continue; }    // not a hit of this call
      const int li = g.plan_layers[p0 + s];
      const LayerDev L = g.layers[li];
      Hit H; load_hit_t<PLANES>(H, a.hits, hid);
      const unsigned rc = step_to_layer(S, nf == 0, a.cov, n, (size_t)i, L, qk * g.bz_layer[li], p.graze_cos_min, mflags, false);
      if (rc) { stat |= rc; stopped = true; continue; }
      SInv o; float c2;
      hit_to_local(S, H, o);
      if (!kalman_update(S, o, c2)) {                          // state untouched by the failed update, but already
        stat |= ST_S_NOT_PD; stop_at = s; redo = true; stopped = true; continue;   // propagated: re-run up to the step before
      }
      if (check && (!state_finite(S) || !(fabsf(c2) <= 3.0e38f))) { stat |= ST_NAN; stop_at = s; redo = true; stopped = true; continue; }
      c2tot += c2; nf++;
    }
    if (redo) continue;
    if (pass == 0 && nf > 0 && (!state_finite(S) || !(fabsf(c2tot) <= 3.0e38f))) continue;
    break;
  }
  if (nf > 0) store_state(S, a.par_out, a.cov_out, n, (size_t)i);
  else copy_seed(a.par, a.cov, a.par_out, a.cov_out, n, (size_t)i);
  a.chi2[i] = c2tot; a.nfit[i] = nf; a.status[i] = stat;
}

// ---- backward fit of one track (reading R7) ---------------------------------------------------------
// Seeds are states on the layer of each track's LAST hit. Hits are taken from the last to the first: give back the
// material of the layer being left, propagate backward (s <= 0), transport, update. After the innermost hit that
// layer's material is given back too (done on the covariance at the output boundary), so the result is the state
// before it. A failing step stops the track, which keeps the state after its last good update.
struct TagTrue { static constexpr bool value = true; };
struct TagFalse { static constexpr bool value = false; };

template <bool STRAG, bool PLANES>
MKF_HD void fit_one_backward(const GeomDev& g, const ParamsDev& p, const FitArgs& a, int i) {
  const int mflags = STRAG ? p.material_flags : (p.material_flags & 3);
  const size_t n = (size_t)a.ld;
  const int pl = a.plan[i];
  if ((unsigned)pl >= (unsigned)g.n_plans) {
    copy_seed(a.par, a.cov, a.par_out, a.cov_out, n, (size_t)i);
    a.chi2[i] = 0.f; a.nfit[i] = 0; a.status[i] = ST_TRUNC;
    return;
  }
  const int p0 = g.plan_off[pl];
  int plen = g.plan_off[pl + 1] - p0;
  if (plen > a.max_plan_len) plen = a.max_plan_len;
 const float qk = -(float)a.q[i] * KAPPA;
  unsigned stat = 0;
  int stop_at = -1;                                              // steps <= stop_at are not processed
  KState S;
  float c2tot; int nf, prev;
  for (int pass = 0; pass < 3; pass++) {
    const bool check = pass == 1;
    load_params(S, a.par, n, (size_t)i);
    c2tot = 0.f; nf = 0; prev = -1;
    bool redo = false, stopped = false;
    // One step: the hit `hid` of plan step s. FIRST: the track's first hit of this pass (6x6 transport of the seed
    // covariance and its factorisation) -- a separate instance, run by all lanes of the warp together before the loop
    // (each at its own step): 10 % of the helices of configs[1] curl before the outer layers, the tracks of a warp met
    // their first hit at 3.3 different steps of the loop, and the warp ran that long branch as often at a third of its lanes.
    auto step = [&](int s, int hid, auto first_tag) {
      constexpr bool FIRST = decltype(first_tag)::value;
      if (hid >= a.hits.n_hits) { stat |= ST_TRUNC; stopped = true; return; }
      const int li = g.plan_layers[p0 + s];
      const LayerDev& L = g.layers[li];
      Hit H; load_hit_t<PLANES>(H, a.hits, hid);
      Prop P;
      float J = 1.f, th02 = 0.f, q4 = 0.f, ipt_old = S.ipt;
      if (!FIRST) {                                            // give back the material of the layer being left
        const LayerDev& Lp = g.layers[prev];
        float rp;
        material_scalars<-1>(Lp.xx0, incidence_of(S), S.ipt, S.sth, mflags, rp, J, th02, q4);
        S.ipt = ipt_old * rp;                                  // the geometry uses the momentum after the give-back
      }
      const unsigned rc = propagate_geom<-1>(S, L, qk * g.bz_layer[FIRST ? li : prev], p.graze_cos_min, 0, false, P);     // R13: back along the arc of the layer being left
      if (rc) { S.ipt = ipt_old; stat |= rc; stopped = true; return; }
      if (FIRST) { float c[21]; load_cov(c, a.cov, n, (size_t)i); commit_first(S, c, P, 0); }
      else commit_step_backward(S, P, J, th02, q4, mflags);
      SInv o; float c2;
      hit_to_local(S, H, o);
      if (!kalman_update(S, o, c2)) { stat |= ST_S_NOT_PD; stop_at = s; redo = true; stopped = true; return; }
      if (check && (!state_finite(S) || !(fabsf(c2) <= 3.0e38f))) { stat |= ST_NAN; stop_at = s; redo = true; stopped = true; return; }
      c2tot += c2; nf++; prev = li;
    };
    const int* th0 = a.track_hits + i;
    const int lo = stop_at;                                      // (stop_at changes when a step fails)
    int sf = lo;                                                 // the track's last hit above lo (independent loads)
    for (int t = lo + 1; t < plen; t++) if (th0[(size_t)t * n] >= 0) sf = t;
    if (sf > lo) step(sf, th0[(size_t)sf * n], TagTrue());
    // no `continue` / `break` out of the layer loop: threads that ran ahead would never rejoin the others (measured: 3x
    // the instructions); the body is a plain if-region, so the warp reconverges after every layer
    const int* th = a.track_hits + (size_t)(plen - 1) * n + i;
    int hid_next = plen - 1 > lo ? *th : -1;                    // the hit id is fetched one step ahead
    for (int s = plen - 1; s > lo; s--) {
      const int hid = hid_next;
      th -= n;
      hid_next = s - 1 > lo ? *th : -1;
      if (hid >= 0 && s < sf && !stopped) step(s, hid, TagFalse());
    }
    if (redo) continue;
    if (pass == 0 && nf > 0 && (!state_finite(S) || !(fabsf(c2tot) <= 3.0e38f))) continue;
    break;
  }
  if (nf > 0) {
    float l[15], c[21];
    ud_to_cov(S.u, S.d, l);
    if (stat == 0) {                                             // give back the innermost layer's material
      const LayerDev& Lp = g.layers[prev];
      float rp, J, th02, q4;
      material_scalars<-1>(Lp.xx0, incidence_of(S), S.ipt, S.sth, mflags, rp, J, th02, q4);
      S.ipt *= rp;
#pragma unroll
      for (int k = 0; k < 5; k++) l[LI(1, k)] *= (k == 1 ? J * J : J);
      l[LI(1, 1)] += q4;
      if (mflags & 1) {
        const float g3 = -S.ipt * fast_div(S.cth, S.sth), g2 = fast_rcp(S.sth);
        l[LI(1, 1)] += g3 * g3 * th02; l[LI(2, 1)] += g3 * th02; l[LI(2, 2)] += th02; l[LI(0, 0)] += g2 * g2 * th02;
      }
    }
    cov_from_local(l, S.f, c);
    a.par_out[i] = S.x + S.xl; a.par_out[n + i] = S.y + S.yl; a.par_out[2 * n + i] = S.z + S.zl;
    a.par_out[3 * n + i] = S.ipt; a.par_out[4 * n + i] = wrap_phi(S.phi); a.par_out[5 * n + i] = S.th;
#pragma unroll
    for (int k = 0; k < 21; k++) a.cov_out[(size_t)k * n + i] = c[k];
  } else copy_seed(a.par, a.cov, a.par_out, a.cov_out, n, (size_t)i);
  a.chi2[i] = c2tot; a.nfit[i] = nf; a.status[i] = stat;
}

}  // namespace mkf

// ---- two-filter smoother of one track (reading R14) ---------------------------------------------------
// Forward filter as fit_one, keeping the PREDICTED state of every fitted hit (propagated, material applied, hit not yet
// used) in the workspace; backward filter (R7) over the fitted hits, seeded with the forward result and D x 1e4; at each
// hit the weighted mean of the stored prediction and the backward filtered state, taken in the local frame of the
// forward point. The combination runs in double (a 5x5 Cholesky per hit; the filters stay in fp32).
namespace mkf {

struct SmoothArgs {
  FitArgs f;                   // par_out / cov_out unused
  float* par_s;                // [mpl][6][ld]
  float* cov_s;                // [mpl][21][ld]
  float* ws;                   // [24][mpl][ld] predicted states
};

constexpr int SM_NF = 24;      // x, y, z, xl, yl, zl, ipt, phi, th, u[10], d[5]

MKF_HD void ud_to_cov_d(const float* u, const float* d, double* p) {
#pragma unroll
  for (int i = 0; i < 5; i++)
#pragma unroll
    for (int j = 0; j <= i; j++) {
      double acc = (i == j ? (double)d[i] : (double)u[UI(j, i)] * (double)d[i]);
#pragma unroll
      for (int k = i + 1; k < 5; k++) acc += (double)u[UI(i, k)] * (double)d[k] * (double)u[UI(j, k)];
      p[LI(i, j)] = acc;
    }
}

// Smoothed state from the stored forward prediction fw[SM_NF] (on a surface of `kind`) and the backward filtered state
// Sb. Local order (phi, ipt, theta, w2, w1). Returns false if P_f + P_b is not positive definite.
MKF_HD bool smooth_combine_dev(const float* fw, int kind, const KState& Sb, float* par6, float* c21) {
  const double xf = (double)fw[0] + (double)fw[3], yf = (double)fw[1] + (double)fw[4], zf = (double)fw[2] + (double)fw[5];
  double cbf = 1.0, sbf = 0.0;
  if (kind == 0) { const double ir = 1.0 / sqrt(xf * xf + yf * yf); cbf = xf * ir; sbf = yf * ir; }
  double Pf[15], Pb[15];
  ud_to_cov_d(fw + 9, fw + 19, Pf);
  ud_to_cov_d(Sb.u, Sb.d, Pb);
  if (kind == 0) {                                               // the backward frame seen from the forward one
    const double cosd = cbf * (double)Sb.f.cb + sbf * (double)Sb.f.sb;
#pragma unroll
    for (int k = 0; k < 4; k++) Pb[LI(4, k)] *= cosd;
    Pb[LI(4, 4)] *= cosd * cosd;
  }
  const double dx = ((double)Sb.x - (double)fw[0]) + ((double)Sb.xl - (double)fw[3]);
  const double dy = ((double)Sb.y - (double)fw[1]) + ((double)Sb.yl - (double)fw[4]);
  const double dz = ((double)Sb.z - (double)fw[2]) + ((double)Sb.zl - (double)fw[5]);
  double a[5];
  const double TWO_PI = 6.283185307179586;
  double dphi = (double)Sb.phi - (double)fw[7];
  dphi -= TWO_PI * rint(dphi / TWO_PI);
  a[0] = dphi; a[1] = (double)Sb.ipt - (double)fw[6]; a[2] = (double)Sb.th - (double)fw[8];
  if (kind == 0) { a[3] = dz; a[4] = cbf * dy - sbf * dx; } else { a[3] = dy; a[4] = dx; }
  // M = (Pf + Pb)^-1 by Cholesky
  double L[15], Li[15];
#pragma unroll
  for (int i = 0; i < 5; i++)
#pragma unroll
    for (int j = 0; j <= i; j++) {
      double acc = Pf[LI(i, j)] + Pb[LI(i, j)];
#pragma unroll
      for (int k = 0; k < j; k++) acc -= L[LI(i, k)] * L[LI(j, k)];
      if (i == j) { if (!(acc > 0.0)) return false; L[LI(i, i)] = sqrt(acc); }
      else L[LI(i, j)] = acc / L[LI(j, j)];
    }
#pragma unroll
  for (int i = 0; i < 5; i++) {
    Li[LI(i, i)] = 1.0 / L[LI(i, i)];
#pragma unroll
    for (int j = 0; j < i; j++) {
      double acc = 0.0;
#pragma unroll
      for (int k = j; k < i; k++) acc -= L[LI(i, k)] * Li[LI(k, j)];
      Li[LI(i, j)] = acc * Li[LI(i, i)];
    }
  }
  double M[15];
#pragma unroll
  for (int i = 0; i < 5; i++)
#pragma unroll
    for (int j = 0; j <= i; j++) {
      double acc = 0.0;
#pragma unroll
      for (int k = i; k < 5; k++) acc += Li[LI(k, i)] * Li[LI(k, j)];
      M[LI(i, j)] = acc;
    }
  double K[5][5];
#pragma unroll
  for (int i = 0; i < 5; i++)
#pragma unroll
    for (int j = 0; j < 5; j++) {
      double acc = 0.0;
#pragma unroll
      for (int k = 0; k < 5; k++) acc += Pf[LI(i, k)] * M[LI(k, j)];
      K[i][j] = acc;
    }
  double as[5];
#pragma unroll
  for (int i = 0; i < 5; i++) {
    double acc = 0.0;
#pragma unroll
    for (int k = 0; k < 5; k++) acc += K[i][k] * a[k];
    as[i] = acc;
  }
  float l[15];
#pragma unroll
  for (int i = 0; i < 5; i++)
#pragma unroll
    for (int j = 0; j <= i; j++) {
      double s1 = 0.0, s2 = 0.0;                                 // P_s = P_f M P_b, symmetrised
#pragma unroll
      for (int k = 0; k < 5; k++) { s1 += K[i][k] * Pb[LI(k, j)]; s2 += K[j][k] * Pb[LI(k, i)]; }
      l[LI(i, j)] = (float)(0.5 * (s1 + s2));
    }
  Frame ff; ff.kind = kind; ff.cb = (float)cbf; ff.sb = (float)sbf;
  cov_from_local(l, ff, c21);
  double xs = xf, ys = yf, zs = zf;
  if (kind == 0) { xs -= sbf * as[4]; ys += cbf * as[4]; zs += as[3]; } else { xs += as[4]; ys += as[3]; }
  par6[0] = (float)xs; par6[1] = (float)ys; par6[2] = (float)zs;
  par6[3] = (float)((double)fw[6] + as[1]); par6[4] = wrap_phi((float)((double)fw[7] + as[0])); par6[5] = (float)((double)fw[8] + as[2]);
  return true;
}

MKF_HD void fit_smooth_one(const GeomDev& g, const ParamsDev& p, const SmoothArgs& sa, int i) {
  const FitArgs& a = sa.f;
  const size_t n = (size_t)a.ld;
  const int mpl = a.max_plan_len;
  const int pl = a.plan[i];
  if ((unsigned)pl >= (unsigned)g.n_plans) { a.chi2[i] = 0.f; a.nfit[i] = 0; a.status[i] = ST_TRUNC; return; }
  const int p0 = g.plan_off[pl];
  const int plen = min(g.plan_off[pl + 1] - p0, mpl);
  const float qk = -(float)a.q[i] * KAPPA;
  unsigned stat = 0;
  KState S;
  load_params(S, a.par, n, (size_t)i);
  float c2tot = 0.f; int nf = 0, last_s = -1; bool smoothable = true;
  // Both layer loops run over the plan steps for the whole warp, their bodies plain if-regions (no `continue` / `break`:
  // a thread that leaves a loop early runs ahead of its warp, alone, and the warp does the rest of its work twice).
  bool stopped = false;
  int hid_next = plen > 0 ? a.track_hits[i] : -1;                // ids one step ahead, the hit before the propagation:
  for (int s = 0; s < plen; s++) {                               // their latency overlaps the arithmetic
    const int hid = hid_next;
    hid_next = s + 1 < plen ? a.track_hits[(size_t)(s + 1) * n + i] : -1;
    if (hid >= 0 && !stopped) do {
      if (hid >= a.hits.n_hits) { stat |= ST_TRUNC; stopped = true; break; }
      Hit H; load_hit(H, a.hits, hid);
      const int li = g.plan_layers[p0 + s];
      const LayerDev& L = g.layers[li];
      const unsigned rc = step_to_layer(S, nf == 0, a.cov, n, (size_t)i, L, qk * g.bz_layer[li], p.graze_cos_min, p.material_flags, false);
      if (rc) { stat |= rc; stopped = true; break; }
      float* w = sa.ws + (size_t)s * n + i;
      const size_t st = (size_t)mpl * n;
      w[0] = S.x; w[st] = S.y; w[2 * st] = S.z; w[3 * st] = S.xl; w[4 * st] = S.yl; w[5 * st] = S.zl;
      w[6 * st] = S.ipt; w[7 * st] = S.phi; w[8 * st] = S.th;
#pragma unroll
      for (int k = 0; k < 10; k++) w[(9 + k) * st] = S.u[k];
#pragma unroll
      for (int k = 0; k < 5; k++) w[(19 + k) * st] = S.d[k];
      SInv o; float c2;
      hit_to_local(S, H, o);
      if (!kalman_update(S, o, c2)) { stat |= ST_S_NOT_PD; smoothable = false; stopped = true; break; }
      if (!state_finite(S) || !(fabsf(c2) <= 3.0e38f)) { stat |= ST_NAN; smoothable = false; stopped = true; break; }
      c2tot += c2; nf++; last_s = s;
    } while (0);
  }
  a.chi2[i] = c2tot; a.nfit[i] = nf;
  bool ok = smoothable && nf > 0;
  const bool had = ok;
  {
#pragma unroll
    for (int k = 0; k < 5; k++) S.d[k] *= 1e4f;                  // the backward filter starts from a weak prior
    int prev = -1;
    hid_next = plen > 0 ? a.track_hits[(size_t)(plen - 1) * n + i] : -1;
    for (int s = plen - 1; s >= 0; s--) {
      const int hid = hid_next;
      hid_next = s > 0 ? a.track_hits[(size_t)(s - 1) * n + i] : -1;
      if (ok && s <= last_s && hid >= 0) do {
        Hit H; load_hit(H, a.hits, hid);
        const int li = g.plan_layers[p0 + s];
        const LayerDev& L = g.layers[li];
        float J = 1.f, th02 = 0.f, q4 = 0.f;
        if (prev >= 0) {
          const LayerDev& Lp = g.layers[prev];
          float rp;
          material_scalars<-1>(Lp.xx0, incidence_of(S), S.ipt, S.sth, p.material_flags, rp, J, th02, q4);
          S.ipt *= rp;
        }
        Prop P;
        const unsigned rc = propagate_geom<-1>(S, L, qk * g.bz_layer[prev >= 0 ? prev : li], p.graze_cos_min, 0, false, P);
        if (rc) { stat |= rc; ok = false; break; }
        commit_step_backward(S, P, J, th02, q4, p.material_flags);
        SInv o; float c2;
        hit_to_local(S, H, o);
        if (!kalman_update(S, o, c2)) { stat |= ST_S_NOT_PD; ok = false; break; }
        if (!state_finite(S) || !(fabsf(c2) <= 3.0e38f)) { stat |= ST_NAN; ok = false; break; }
        float fw[SM_NF];
        const size_t st = (size_t)mpl * n;
        const float* w = sa.ws + (size_t)s * n + i;
#pragma unroll
        for (int k = 0; k < SM_NF; k++) fw[k] = w[k * st];
        float par6[6], c21[21];
        if (!smooth_combine_dev(fw, L.kind, S, par6, c21)) { stat |= ST_S_NOT_PD; ok = false; break; }
#pragma unroll
        for (int k = 0; k < 6; k++) sa.par_s[((size_t)s * 6 + k) * n + i] = par6[k];
#pragma unroll
        for (int k = 0; k < 21; k++) sa.cov_s[((size_t)s * 21 + k) * n + i] = c21[k];
        prev = li;
      } while (0);
    }
    if (had && !ok)                                              // not smoothed: every state of the track is zero
      for (int s = 0; s < mpl; s++) {
        for (int k = 0; k < 6; k++) sa.par_s[((size_t)s * 6 + k) * n + i] = 0.f;
        for (int k = 0; k < 21; k++) sa.cov_s[((size_t)s * 21 + k) * n + i] = 0.f;
      }
  }
  a.status[i] = stat;
}

}  // namespace mkf
