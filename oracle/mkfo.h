/* mkfo.h — C ABI of the ORACLE (test infrastructure, not the product).
 *
 * Plain, slow, float64 CPU restatement of the mkFit-style Kalman-filter hot path described in
 * /root/reference/PAPER.md (arxiv 2002.06295): propagate a track state layer to layer, update it with a
 * hit (§1), on a lightweight geometry of barrel layers at average r and forward layers at
 * average z with 3D hits (§2), combinatorial building with a per-seed cap on cloned
 * candidates, short-track preservation and duplicate removal (abstract).
 * The paper prints no formulas (PAPER.md:29 defers to its refs [3-12]); every formula here follows the
 * readings C1..C10 / U1..U22 listed in DESIGN.md §3, and is pinned by tests/test_oracle_*.py.
 *
 * ONLY tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this
 * library. It shares no code, header, table or constant with paper_2002_06295_b200/csrc/.
 *
 * All pointers are HOST pointers. Inputs are the same fp32 arrays the CUDA library takes, widened exactly
 * to double; all arithmetic and all outputs are double. Arrays are SoA, plane-major: par[k*n+i],
 * cov[k*n+i] with k = i*(i+1)/2+j (j<=i) packed lower triangle of the 6x6 covariance.
 * State u = (x, y, z, ipt, phi, theta): cm, 1/GeV, rad; charge q = +-1 separately. */
#ifndef MKFO_H
#define MKFO_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct { int kind;            /* 0 barrel cylinder, 1 disk */
                 float pos;           /* r (barrel) or signed z (disk) */
                 float lo, hi;        /* barrel: zmin,zmax ; disk: rmin,rmax */
                 float xx0;           /* thickness in radiation lengths at normal incidence */
                 float eta_lo, eta_hi;/* hit pseudorapidity range spanned by the eta bins */ } mkfo_layer;
typedef struct { int n_layers; const mkfo_layer* layers; float bz; int n_phi_bins, n_eta_bins;
                 int n_plans; const int* plan_off; const int* plan_layers;
                 const float* bz_layer; /* R13 field hook: Bz of the step that ENDS on layer l (NULL: bz everywhere) */ } mkfo_geometry;
typedef struct { float chi2_cut; int max_cand; int max_consec_miss; int min_hits_keep;
                 float score_hit, score_miss; float graze_cos_min; int material_flags; /* 1 MS, 2 dE/dx, 4 energy-loss straggling (R12) */
                 float dup_frac; } mkfo_params;
typedef struct { int n_events; int n_hits; const int* layer_off; /* [n_events*(n_layers+1)] */
                 const float *x, *y, *z; const float* V; /* V[6][n_hits]: xx,xy,yy,xz,yz,zz */ } mkfo_hits;

enum { MKFO_PROP_UNREACHABLE = 1, MKFO_GRAZING = 2, MKFO_S_NOT_PD = 4, MKFO_NAN = 8,
       MKFO_STOPPED_ELOSS = 16, MKFO_TRUNCATED = 32 };

/* ---- single-step functions (exported so the pins can reach every formula) ------------------------ */
/* C1-C4: propagate u (6) with full 6x6 covariance C (36, row-major, may be NULL) to a surface.
 * kind 0: cylinder r=pos; kind 1: plane z=pos. Outputs u1 (6), F (36, may be NULL), C1 (36, may be NULL),
 * s (transverse path). Returns 0 or MKFO_PROP_UNREACHABLE. */
int mkfo_propagate(int kind, double pos, double bz, int q, const double* u, const double* C,
                   double* u1, double* F, double* C1, double* s);
/* C1 alone: helix step by transverse path s. */
void mkfo_helix_step(double bz, int q, const double* u, double s, double* u1);
/* C5: material at a layer (state already on the surface). In/out u (6), C (36). Returns 0 or STOPPED_ELOSS.
 * theta0_out / dE_out (may be NULL) receive the Highland angle and the energy loss. */
int mkfo_material(int kind, double xx0, int flags, double* u, double* C, double* theta0_out, double* dE_out);
/* R7: the same with a direction: dir = +1 as above, dir = -1 backward (s <= 0; energy given back). */
int mkfo_propagate_dir(int kind, double pos, double bz, int q, int dir, const double* u, const double* C,
                       double* u1, double* F, double* C1, double* s);
int mkfo_material_dir(int kind, double xx0, int flags, int dir, double* u, double* C, double* theta0_out, double* dE_out);
/* Bethe-Bloch -dE/dx [GeV/cm] in silicon for a pion of momentum p [GeV]; Highland theta0 for thickness t. */
double mkfo_dedx(double p);
/* R12: variance [GeV^2] of the energy lost in silicon of thickness t (radiation lengths along the path) by a pion of
 * momentum p: xi Tmax (1 - beta^2 / 2), xi = (K/2)(Z/A) rho t X0 / beta^2 (Gaussian straggling). */
double mkfo_straggling_var(double p, double t);
double mkfo_highland(double p, double t);
/* C6: chi2 of hit m (3) with covariance V (6: xx,xy,yy,xz,yz,zz); returns 0 or S_NOT_PD. */
int mkfo_chi2(const double* u, const double* C, const double* m, const double* V, double* chi2);
/* C6: Kalman update (Joseph form). In/out u, C. */
int mkfo_update(double* u, double* C, const double* m, const double* V, double* chi2);
/* U11: search window of a propagated state on layer L. Outputs eta-bin range [e0,e1] and phi-bin range
 * [p0, p0+np) (np<=n_phi, wraps). vmax = (v_xy, v_zz) of the layer's hits. */
void mkfo_window(const mkfo_geometry* g, const mkfo_params* p, int layer, const double* u, const double* C,
                 const double* vmax, int* e0, int* e1, int* p0, int* np);

/* ---- the four calls named by BASELINE.json north_star -------------------------------------------- */
/* C8. bin_off [n_events*n_layers*n_phi*n_eta + 1], sorted_id [n_hits], vmax [n_events*n_layers*2]. */
int mkfo_build_hit_index(const mkfo_geometry*, const mkfo_hits*, unsigned* bin_off, int* sorted_id, float* vmax);
/* R9: hits with mask[i] != 0 are left out (mask may be NULL) */
int mkfo_build_hit_index_masked(const mkfo_geometry*, const mkfo_hits*, const unsigned char* mask, unsigned* bin_off,
                                int* sorted_id, float* vmax);
/* R9: mask[h] = 1 for the hits of high-quality tracks */
int mkfo_mask_hits(int n, int n_hits, const int* hit_ids, int max_plan_len, const int* nhits, const float* chi2,
                   const unsigned char* keep, int min_hits, float max_chi2_ndf, unsigned char* mask);
/* C7. seeds par[6][n] cov[21][n] (fp32), q[n]; plan[n]; track_hits[max_plan_len][n] (global hit id or <0).
 * Outputs (double) par_out[6][n], cov_out[21][n], chi2[n], nfit[n], status[n]. */
int mkfo_fit(const mkfo_geometry*, const mkfo_params*, const mkfo_hits*, int n, const float* par,
             const float* cov, const signed char* q, const signed char* plan, const int* track_hits,
             int max_plan_len, double* par_out, double* cov_out, double* chi2, int* nfit, unsigned* status);
/* R14 (SURVEY f1 "backward fit + smoother"; "Fitting simply applies the KF procedure to all hits").
 * Two-filter smoother. Forward filter as mkfo_fit, keeping at every fitted hit k the PREDICTED state (propagated, the
 * layer's material applied, hit k not yet used: hits 0..k-1). Backward filter (R7) over the fitted hits, seeded with the
 * forward result at the last fitted hit, covariance x 1e4 (a prior worth 1e-4 of the data); at hit k its FILTERED state
 * (hits k..last) describes the same place: the outer side of layer k. Smoothed state at hit k = their weighted mean,
 * taken in the local frame of the forward point (in-surface 1, in-surface 2, ipt, phi, theta): a = T (u_b - u_f),
 * M = (P_f + P_b)^-1, a_s = P_f M a, P_s = P_f M P_b (symmetrised); u_s = u_f + T^T a_s, C_s = T^T P_s T.
 * par_s[max_plan_len][6][n], cov_s[max_plan_len][21][n]: smoothed state per plan step (zero where the step has no
 * fitted hit); chi2 / nfit / status: those of the forward filter. A track whose forward filter fails at an update
 * (S not PD, NaN) or whose backward filter fails anywhere is not smoothed (all zero, status says why). */
int mkfo_fit_smooth(const mkfo_geometry*, const mkfo_params*, const mkfo_hits*, int n, const float* par,
             const float* cov, const signed char* q, const signed char* plan, const int* track_hits,
             int max_plan_len, double* par_s, double* cov_s, double* chi2, int* nfit, unsigned* status);
/* The combination step alone (for the pins): forward (u_f, C_f) and backward (u_b, C_b) on a surface of `kind`. */
int mkfo_smooth_combine(int kind, const double* u_f, const double* C_f, const double* u_b, const double* C_b,
             double* u_s, double* C_s);
/* R7. Backward fit: seeds are states on the layer of each track's LAST hit; hits are processed from the last to the
 * first; output = state at the innermost hit before that layer's material. Same arguments as mkfo_fit. */
int mkfo_fit_backward(const mkfo_geometry*, const mkfo_params*, const mkfo_hits*, int n, const float* par,
             const float* cov, const signed char* q, const signed char* plan, const int* track_hits,
             int max_plan_len, double* par_out, double* cov_out, double* chi2, int* nfit, unsigned* status);
/* C9. brute_force!=0: every hit of the layer is tried (small events); else the binned window search.
 * hit_ids [max_plan_len][n]: id | -1 miss | -2 not crossed. margin[n]: smallest decision margin met (U20).
 * n_chi2_evals (may be NULL): number of (candidate,hit) chi2 evaluations done. */
int mkfo_build_tracks(const mkfo_geometry*, const mkfo_params*, const mkfo_hits*, const unsigned* bin_off,
             const int* sorted_id, const float* vmax, int brute_force, int n, const float* par,
             const float* cov, const signed char* q, const int* seed_event, const int* seed_hits,
             const signed char* plan, int max_plan_len, double* par_out, double* cov_out, double* chi2,
             double* score, int* nhits, int* nmiss, int* hit_ids, unsigned* status, double* margin,
             long long* n_chi2_evals);
/* R15: mkfo_build_tracks with overlap-hit recovery. module[n_hits]: module id per hit;
 * hit_ids2[max_plan_len][n]: the second hit taken on a plan step, or -2. A child that took hit h1 may take one more
 * hit of the same layer from another module: the best (chi2 against the state updated with h1, below the cut) among its
 * parent's N_c best hits of the layer that rank after h1 there (so a pair is made once, by the child of its better hit). nhits, chi2 and score include it. module == NULL: mkfo_build_tracks. */
int mkfo_build_tracks_overlap(const mkfo_geometry*, const mkfo_params*, const mkfo_hits*, const unsigned* bin_off,
             const int* sorted_id, const float* vmax, int brute_force, int n, const float* par,
             const float* cov, const signed char* q, const int* seed_event, const int* seed_hits,
             const signed char* plan, int max_plan_len, double* par_out, double* cov_out, double* chi2,
             double* score, int* nhits, int* nmiss, int* hit_ids, unsigned* status, double* margin,
             long long* n_chi2_evals, const int* module, int* hit_ids2);
/* C10. track_off[n_events+1]; hit_ids[max_plan_len][n]; keep[n], n_kept[n_events]. */
int mkfo_remove_duplicates(const mkfo_params*, int n_events, const int* track_off, const int* hit_ids,
             int max_plan_len, const int* nhits, const float* score, unsigned char* keep, int* n_kept);
/* R8: three-threshold strip clustering. Outputs sized for the worst case (n_strips). */
int mkfo_cluster_strips(int n_modules, const int* module_off, const unsigned short* adc, const float* noise,
                        const unsigned char* bad, float seed_thr, float chan_thr, float clus_thr, int min_charge,
                        int max_holes, int max_bad, int* out_module, int* out_first, int* out_last,
                        unsigned* out_charge, float* out_bary);
int mkfo_num_threads(void);
#ifdef __cplusplus
}
#endif
#endif
