/* mkf.h — C ABI of the B200-native (sm_100a) batched Kalman-filter track fit / track building library.
 *
 * Hot path of arxiv 2002.06295 (mkFit, /root/reference/PAPER.md): "propagate a track state from layer N-1 to
 * layer N, update it with the hit" (§1), on a "lightweight" geometry of barrel layers collapsed at
 * their average r and forward layers at their average z, relying on 3D hit positions (§2), with
 * combinatorial building where "only the best ranking [candidates] are cloned at each layer (with a per-seed
 * cap)", short-track preservation and explicit duplicate removal (PAPER.md:5 abstract), and a
 * fit that "applies the KF procedure to all hits identified during building". The paper prints
 * no formulas (PAPER.md:29 defers to its refs); the formulas are the readings C1..C10 / U1..U22 of DESIGN.md §3.
 *
 * CONVENTIONS
 *  - Every data pointer of the mkf_* calls below is a DEVICE pointer into caller-owned memory unless marked
 *    "host". The *_host entry points take HOST pointers for everything and stage through device memory
 *    themselves. The library never frees or keeps caller memory after a call returns.
 *  - Calls enqueue work on `stream` (a cudaStream_t passed as void*, NULL = default stream) and do NOT
 *    synchronise (the *_host entry points do synchronise before returning). Outputs are valid after the
 *    caller synchronises the stream.
 *  - Scratch comes from a caller-provided device workspace `ws` of at least mkf_workspace_bytes(...) bytes,
 *    256-byte aligned. Its contents are undefined between calls.
 *  - Arrays are SoA, plane-major: par[k*n + i] (k = 0..5: x, y, z [cm], ipt = 1/pT [1/GeV], phi, theta [rad]);
 *    cov[k*n + i] with k = a*(a+1)/2 + b (b <= a) the packed lower triangle of the symmetric 6x6 covariance.
 *    The charge q = +-1 is carried separately. Field: uniform Bz [T]; kappa = 0.0029979246 GeV/(T cm).
 *  - Return value: MKF_OK or a negative error code. Numerical trouble is never an error code: it is reported
 *    per track in `status` (bit set below). mkf_last_error(ctx) gives a text for the last failing call.
 *  - All arithmetic is fp32 (positions carried as an unevaluated sum of two floats inside the kernels; the hit
 *    bin keys are evaluated in fp64, reading U12). No host fallback exists: without a CUDA device every compute
 *    call returns MKF_CUDA_ERROR. */
#ifndef MKF_H
#define MKF_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { MKF_OK = 0, MKF_INVALID_ARG = -1, MKF_CUDA_ERROR = -2, MKF_WORKSPACE_TOO_SMALL = -3, MKF_UNSUPPORTED = -4 };

/* per-track status bits */
enum { MKF_PROP_UNREACHABLE = 1, /* next surface not reachable going forward with < half a turn (U5, U6) */
       MKF_GRAZING = 2,          /* incidence too shallow: cos(alpha) < graze_cos_min (barrel), |cos theta| < 0.05 (disk) (U7) */
       MKF_S_NOT_PD = 4,         /* residual covariance S = C(0:3,0:3)+V not positive definite (C6) */
       MKF_NAN = 8,              /* non-finite value after an update */
       MKF_STOPPED_ELOSS = 16,   /* energy exhausted by dE/dx (C5) */
       MKF_TRUNCATED = 32 };     /* building: nothing with >= min_hits_keep hits; the seed itself is returned. Also set on a
                                    track whose plan id, event id or a hit id lies outside the ranges of the call */

enum { MKF_MAX_LAYERS = 64, MKF_MAX_PLANS = 8, MKF_MAX_PLAN_STEPS = 192 /* total over plans */, MKF_MAX_CAND = 8 };

/* workspace query ids */
enum { MKF_CALL_BUILD_HIT_INDEX = 0, MKF_CALL_FIT = 1, MKF_CALL_BUILD_TRACKS = 2, MKF_CALL_REMOVE_DUPLICATES = 3,
       MKF_CALL_CLUSTER_STRIPS = 4 /* n_hits = number of strips, n_seeds = capacity */,
       MKF_CALL_FIT_SMOOTH = 5 /* n_seeds = number of tracks; for max_plan_len = mkf_max_plan_len(ctx) */,
       MKF_CALL_BUILD_TRACKS_OVERLAP = 6 };

typedef struct mkf_ctx mkf_ctx;       /* opaque: geometry, parameters, last error text */

/* One detector layer of the lightweight geometry. */
typedef struct { int kind;            /* 0 barrel cylinder, 1 disk */
                 float pos;           /* r (barrel) or signed z (disk) [cm] */
                 float lo, hi;        /* acceptance: barrel zmin,zmax ; disk rmin,rmax [cm] */
                 float xx0;           /* thickness in radiation lengths at normal incidence */
                 float eta_lo, eta_hi;/* hit pseudorapidity range spanned by the eta bins (U16) */ } mkf_layer;

/* Geometry: all pointers HOST, copied by mkf_create. A "plan" is the ordered list of layers a seed is
 * followed through (U17); plan p = plan_layers[plan_off[p] .. plan_off[p+1]). */
typedef struct { int n_layers; const mkf_layer* layers; float bz; int n_phi_bins, n_eta_bins;
                 int n_plans; const int* plan_off; const int* plan_layers;
                 const float* bz_layer; /* field hook (reading R13; "geometry, material, magnetic field"):
                                           [n_layers] Bz [T] of the step that ENDS on layer l (a backward step runs in the
                                           field of the layer it leaves); NULL: bz everywhere */ } mkf_geometry;

typedef struct { float chi2_cut;      /* hit accepted iff chi2 < chi2_cut (30) */
                 int max_cand;        /* live candidates kept per seed per layer, <= MKF_MAX_CAND (6 or 8) */
                 int max_consec_miss; /* a candidate stops at this many consecutive missed layers (2) */
                 int min_hits_keep;   /* stopped candidates with at least this many hits are preserved (4) */
                 float score_hit, score_miss; /* score = score_hit*nhits - score_miss*nmiss - chi2 (U13) */
                 float graze_cos_min; /* U7 (0.25) */
                 int material_flags;  /* bit0 multiple scattering, bit1 dE/dx (C5), bit2 energy-loss straggling (R12; needs bit1) */
                 float dup_frac;      /* duplicate if shared/min(nhits) > dup_frac (0.5) */ } mkf_params;

/* Hits of n_events events, grouped by (event, layer): the hits of (ev, l) are the ids
 * layer_off[ev*(n_layers+1)+l] .. layer_off[ev*(n_layers+1)+l+1]; ids are global (0..n_hits).
 * rec (may be NULL): the same hits as 48-byte records rec[12*id .. 12*id+11] = {x, y, z, Vxx | Vxy, Vyy, Vxz, Vyz |
 * Vzz, 0, 0, 0}, 16-byte aligned, written by mkf_pack_hits (or by the caller). The SoA planes serve streaming
 * access in id order (36 B per hit); a gather by scattered hit id (a fit over hit lists that are not sorted, the
 * update step of the building) costs 9 sectors = 288 B per hit on the planes and 2 sectors = 64 B on a record, so
 * every kernel that gathers by id reads `rec` when it is given. x, y, z, V must be valid in either case. */
typedef struct { int n_events; int n_hits; const int* layer_off;
                 const float *x, *y, *z; const float* V; /* V[6][n_hits]: xx,xy,yy,xz,yz,zz */
                 const float* rec;
                 const int* module; /* [n_hits] detector module of each hit, or NULL. Only overlap-hit recovery reads it
                                       (mkf_build_tracks_overlap); mkf_build_hit_index copies it into the packed records. */
               } mkf_hits;

/* The phi/eta-binned hit index (C8), written by mkf_build_hit_index, read by mkf_build_tracks.
 * bin_off  [n_events*n_layers*n_phi*n_eta + 1]  exclusive prefix of hits per bin (bin = ie*n_phi + ip inside
 *          segment (ev*n_layers + l)), last entry = n_hits;
 * sorted_id[n_hits]  hit ids ordered by (segment, bin, id);
 * vmax     [n_events*n_layers*2]  per segment: max over hits of the larger eigenvalue of the xy block of V, max V_zz;
 * packed   [n_hits*12 + 4]  the hits in sorted order, as a block of n_hits 16-byte positions {x,y,z,id(bits)} followed,
 *          from float 4*(n_hits + (n_hits & 1)) on (so that every record is one 32-byte sector; 256-byte aligned base), by
 *          a block of n_hits 32-byte covariances {Vxx,Vxy,Vyy,Vxz | Vyz,Vzz,module(bits),0} (a derived copy so that a bin scan
 *          reads contiguous memory; may be NULL in mkf_build_hit_index, in which case mkf_build_tracks gathers from
 *          the SoA arrays instead). */
typedef struct { unsigned* bin_off; int* sorted_id; float* vmax; float* packed; } mkf_hit_index;

typedef struct { int n; float* par; float* cov; signed char* q; } mkf_states;   /* par[6][n], cov[21][n], q[n] */

/* ---- context ----------------------------------------------------------------------------------------- */
/* Copies geometry and parameters. Errors: INVALID_ARG (null, n_layers<1), UNSUPPORTED (limits above). */
int mkf_create(mkf_ctx** out, const mkf_geometry* geom, const mkf_params* params);
void mkf_destroy(mkf_ctx*);
const char* mkf_last_error(const mkf_ctx*);
/* Bytes of device workspace the given call needs for these sizes (0 is a valid answer). */
size_t mkf_workspace_bytes(const mkf_ctx*, int call_id, int n_events, int n_hits, int n_seeds);
/* Number of kernel launches the library has enqueued through this context so far. */
long long mkf_launch_count(const mkf_ctx*);
/* Longest plan of the geometry (the leading dimension callers give track_hits / hit_ids). */
int mkf_max_plan_len(const mkf_ctx*);

/* Writes the 48-byte hit records (see mkf_hits.rec) of hits->x,y,z,V to rec_out[12 * n_hits] (device, 16-byte
 * aligned). One streaming pass: 36 B read + 48 B written per hit. hits->rec is ignored. Errors: INVALID_ARG, CUDA_ERROR. */
int mkf_pack_hits(mkf_ctx*, const mkf_hits*, float* rec_out, void* stream);

/* ---- the four calls of BASELINE.json north_star -------------------------------------------------------- */
/* a1 / C8 ("data preparation ... for each event"). Errors: INVALID_ARG, WORKSPACE_TOO_SMALL,
 * UNSUPPORTED (n_hits >= 2^28), CUDA_ERROR. */
int mkf_build_hit_index(mkf_ctx*, const mkf_hits*, mkf_hit_index* out, void* ws, size_t ws_bytes, void* stream);

/* mkf_build_hit_index for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops): same inputs, same outputs (bit-identical), no workspace argument. Its scratch (8 bytes per hit) is a fixed
 * array of 8 MiB inside the library's device image, held by every GPU that loads the library until exit; the call
 * makes no cudaMalloc / cudaFree and calls no allocating routine (the first call on a device resolves the array's
 * address once: make that call outside a capture). Limits: n_hits <= MKF_STATIC_MAX_HITS and at most 16384 bins
 * per layer, else MKF_UNSUPPORTED with nothing launched; no masked variant. All calls on one device share the
 * array: two calls that overlap on the GPU (different streams, no dependency between them) race and give undefined
 * results; calls on one stream, or ordered by events, are safe. The array needs no clearing between calls.
 * Errors: INVALID_ARG, UNSUPPORTED, CUDA_ERROR. */
#define MKF_STATIC_MAX_HITS (1 << 20)
int mkf_build_hit_index_static(mkf_ctx*, const mkf_hits*, mkf_hit_index* out, void* stream);

/* a11 / C7 ("Fitting simply applies the KF procedure to all hits identified during building").
 * seeds: n states; plan[n]: plan id per track; track_hits[max_plan_len][n]: global hit id per plan step or <0.
 * For every step with a hit: propagate (C2/C3) -> grazing test (U7) -> covariance transport (C4) -> material
 * (C5) -> chi2 + update (C6). A track stops at the first failing step and keeps its last good state.
 * out: states after the last fitted hit (phi wrapped to (-pi,pi]); chi2[n] total; nfit[n]; status[n]. */
int mkf_fit(mkf_ctx*, const mkf_hits*, const mkf_states* seeds, const signed char* plan, const int* track_hits,
            int max_plan_len, mkf_states* out, float* chi2, int* nfit, unsigned* status,
            void* ws, size_t ws_bytes, void* stream);

/* SURVEY.md f1 / reading R7 of DESIGN.md: the same filter run from the outermost hit inwards, giving the parameters
 * at the innermost hit ("Fitting simply applies the KF procedure to all hits"). Same arguments as
 * mkf_fit; `seeds` are states on the layer of each track's LAST hit (e.g. mkf_fit's output with the covariance
 * scaled up). Per hit, from the last to the first: give back the material of the layer being left (C5 with the
 * energy loss as a gain), propagate backward (C2/C3 with s <= 0), grazing test, transport, chi2 + update; after the
 * innermost hit that layer's material is given back too, so the output is the state before it. A track stops at its
 * first failing step and keeps the state after its last good update. */
int mkf_fit_backward(mkf_ctx*, const mkf_hits*, const mkf_states* seeds, const signed char* plan, const int* track_hits,
            int max_plan_len, mkf_states* out, float* chi2, int* nfit, unsigned* status,
            void* ws, size_t ws_bytes, void* stream);

/* SURVEY.md f1 / reading R14 of DESIGN.md: two-filter smoother ("Fitting simply applies the KF procedure to
 * all hits"). Same inputs as mkf_fit. Forward filter keeping, at every fitted hit, the predicted state (propagated,
 * material applied, hit not yet used); backward filter over the fitted hits from the forward result with covariance
 * x 1e4; at each hit the weighted mean of the two, in the local frame of the forward point:
 * M = (P_f + P_b)^-1, a_s = P_f M a, P_s = P_f M P_b. The state at plan step s describes the outer side of that layer.
 * par_s[max_plan_len][6][n], cov_s[max_plan_len][21][n]: zero where the step has no fitted hit; chi2, nfit, status: the
 * forward filter's. A track whose forward filter fails at an update, or whose backward filter fails anywhere, is not
 * smoothed (all zero; status says why). ws: mkf_workspace_bytes(ctx, MKF_CALL_FIT_SMOOTH, 0, 0, n) bytes (24 floats per
 * track and plan step); max_plan_len must be mkf_max_plan_len(ctx). */
int mkf_fit_smooth(mkf_ctx*, const mkf_hits*, const mkf_states* seeds, const signed char* plan, const int* track_hits,
            int max_plan_len, float* par_s, float* cov_s, float* chi2, int* nfit, unsigned* status,
            void* ws, size_t ws_bytes, void* stream);

/* a12 / C9. seeds: n states at their first hit; seed_event[n]; seed_hits[3][n] global hit ids;
 * plan[n]. Each seed is first fitted through its own three hits, then followed through the rest of its plan.
 * max_plan_len must be mkf_max_plan_len(ctx). ws: mkf_workspace_bytes(ctx, MKF_CALL_BUILD_TRACKS, n_events, n_hits,
 * n_seeds) bytes (the seeds' fitted states, their processing order and the hit-list trellis live there).
 * out: state of the winning candidate; chi2, score, nhits (incl. seed hits), nmiss;
 * hit_ids[max_plan_len][n]: hit id | -1 missed layer | -2 layer not crossed; status (a seed whose plan or event id
 * is out of range, or whose hits are not on its plan in plan order, comes back unchanged with MKF_TRUNCATED).
 * Limits: n_hits <= 2^28 - 2, at most 255 phi and 255 eta bins (MKF_UNSUPPORTED otherwise).
 * Any scoring parameters are valid: the children of a layer are ranked by the total order U14 whatever the relation of
 * score_hit, score_miss and chi2_cut. */
int mkf_build_tracks(mkf_ctx*, const mkf_hits*, const mkf_hit_index*, const mkf_states* seeds,
            const int* seed_event, const int* seed_hits, const signed char* plan, int max_plan_len,
            mkf_states* out, float* chi2, float* score, int* nhits, int* nmiss, int* hit_ids, unsigned* status,
            void* ws, size_t ws_bytes, void* stream);

/* SURVEY.md f2 / reading R15 of DESIGN.md: mkf_build_tracks with overlap-hit recovery ("the recovery of hits
 * in overlapping detector modules, so that more than one hit per layer can be assigned to tracks"). hits->module must
 * be given (also to mkf_build_hit_index, if its packed records are used). A candidate that took hit h1 on a layer may
 * take ONE more hit of that layer: the best one (chi2 against the state already updated with h1, below chi2_cut) among
 * its parent's max_cand best hits of the layer (by chi2 against the propagated state) that rank after h1 in that list
 * (a pair is then made once, by the child of its better hit), with module[h2] != module[h1]. The state is updated again; chi2, nhits and score include it (an update that does not stay finite is not
 * taken). The ranking of the layer is done on the first hits alone. hit_ids2[max_plan_len][n]: the second hit of each
 * plan step, or -2. ws: mkf_workspace_bytes(ctx, MKF_CALL_BUILD_TRACKS_OVERLAP, n_events, n_hits, n_seeds).
 * mkf_remove_duplicates and mkf_fit keep working on hit_ids (one hit per layer). */
int mkf_build_tracks_overlap(mkf_ctx*, const mkf_hits*, const mkf_hit_index*, const mkf_states* seeds,
            const int* seed_event, const int* seed_hits, const signed char* plan, int max_plan_len,
            mkf_states* out, float* chi2, float* score, int* nhits, int* nmiss, int* hit_ids, int* hit_ids2,
            unsigned* status, void* ws, size_t ws_bytes, void* stream);

/* Work counters of mkf_build_tracks (SURVEY.md §8d asks for candidate-layer-steps/s and chi2 evaluations/s): while
 * `counters` (device, 8 x unsigned long long, zeroed by the caller) is set, every mkf_build_tracks call on this context
 * adds to it: [0] candidate-layer-steps (propagations that landed on a layer), [1] hit positions tested inside windows,
 * [2] chi2 evaluations (hits that passed the position test: their covariance is read), [3] hits accepted (chi2 < cut),
 * [4] Kalman updates, [5..7] reserved. NULL (the default) switches counting off. The counts do not depend on timing
 * and equal the oracle's n_chi2_evals only in order of magnitude (the oracle evaluates chi2 on whole bins). */
int mkf_set_build_counters(mkf_ctx*, unsigned long long* counters);

/* a10 / C10 ("duplicate tracks ... explicitly removed in an additional processing step").
 * track_off[n_events+1] (device): tracks of event ev are track_off[ev]..track_off[ev+1]; n = total tracks (the
 * plane stride of hit_ids); n_hits = size of the hit-id space. keep[n] = 0/1, n_kept[n_events]. */
int mkf_remove_duplicates(mkf_ctx*, int n_events, int n, int n_hits, const int* track_off, const int* hit_ids,
            int max_plan_len, const int* nhits, const float* score, unsigned char* keep, int* n_kept,
            void* ws, size_t ws_bytes, void* stream);

/* ---- SURVEY.md f4 / reading R9 of DESIGN.md: hit masking between iterations ("Hits used in tracks
 * reconstructed with high quality are masked to reduce the combinatorics of the next iteration") ------------------
 * mkf_mask_hits: mask[h] = 1 for every hit (id >= 0) of a high-quality track; other entries are left as they are, so
 * masks accumulate over iterations (the caller zeroes the mask before the first). High quality (R9; the paper gives no
 * definition): keep[i] != 0 (keep == NULL: every track), nhits[i] >= min_hits and chi2[i] <= max_chi2_ndf * (2 nhits[i] - 5),
 * compared in fp32. hit_ids[max_plan_len][n], nhits, chi2, keep as written by mkf_build_tracks / mkf_remove_duplicates.
 * mkf_build_hit_index_masked: mkf_build_hit_index without the hits with mask[i] != 0: they are in no bin and do not
 * count for vmax; sorted_id / packed hold bin_off[last] <= n_hits entries. mask == NULL: the plain index. Same workspace.
 * All pointers device; caller's stream; no synchronisation. */
int mkf_mask_hits(mkf_ctx*, int n, int n_hits, const int* hit_ids, int max_plan_len, const int* nhits, const float* chi2,
            const unsigned char* keep, int min_hits, float max_chi2_ndf, unsigned char* mask, void* stream);
int mkf_build_hit_index_masked(mkf_ctx*, const mkf_hits*, const unsigned char* mask, mkf_hit_index* out,
            void* ws, size_t ws_bytes, void* stream);

/* ---- SURVEY.md f3 / reading R8 of DESIGN.md: strip clustering ------------------------------
 * "seed strips with ADC values greater than 3 times the expected noise are identified; second, clusters are formed
 * adding to the seed all strips with ADC values above twice the expected noise that are either consecutive or have
 * a small gap (the size of the allowed gap depends on the presence of bad strips in the module); finally, the
 * cluster is required to have a quadrature sum of the strip ADCs larger than 5 times the quadrature sum of the
 * expected noise, and to have a minimum total charge."
 * Input: the strips of all modules of all events of the batch, concatenated; module m owns strips
 * module_off[m]..module_off[m+1]-1 (ascending; empty modules allowed). adc: pedestal-subtracted counts; noise: the
 * expected noise of each strip; bad: non-zero = bad strip (never counted, may be bridged). adc and noise must be
 * 16-byte aligned and bad 8-byte aligned; module_off[0] = 0 and module_off[n_modules] = n_strips (not checked: the
 * offsets live on the device); n_strips <= 2^31 - 16384; max_holes + max_bad <= 31 (MKF_UNSUPPORTED otherwise).
 * Output (ordered by module, then first strip): module, first and last strip (index inside the module), charge =
 * sum adc, bary = sum adc (strip + 1/2) / sum adc in strip units. *n_clusters = number of clusters found. With
 * *n_clusters > capacity ONLY *n_clusters is defined (the record arrays then hold an unspecified subset with holes,
 * because records are staged in tile-arrival order): the caller retries with more room. mkf_cluster_strips_host
 * copies no records back in that case. */
typedef struct { float seed_thr, chan_thr, clus_thr; int min_charge, max_holes, max_bad; } mkf_strip_params;
typedef struct {
  int n_modules, n_strips;
  const int* module_off;            /* [n_modules + 1] */
  const unsigned short* adc;        /* [n_strips] */
  const float* noise;               /* [n_strips] */
  const unsigned char* bad;         /* [n_strips] */
} mkf_strips;
typedef struct {
  int capacity;
  int *module, *first, *last;       /* [capacity] */
  unsigned* charge;                 /* [capacity] */
  float* bary;                      /* [capacity] */
  int* n_clusters;                  /* [1] */
} mkf_clusters;
/* Device pointers, caller's stream, no synchronisation. ws: mkf_workspace_bytes(ctx, MKF_CALL_CLUSTER_STRIPS, 0, n_strips, capacity). */
int mkf_cluster_strips(mkf_ctx*, const mkf_strips*, const mkf_strip_params*, const mkf_clusters* out,
            void* ws, size_t ws_bytes, void* stream);

/* ---- host-buffer entry points (end-to-end use: all pointers HOST; synchronous) ------------------------- */
/* Device memory of the host entry points is an arena owned by the context: it grows to the largest call seen and is
 * freed by mkf_destroy, so repeated calls allocate nothing ("a memory pool to pay the allocation overhead
 * only at the beginning and end of job"). Copies are asynchronous (and overlap the kernels) only from pinned host
 * memory; pageable buffers work but are staged by the driver. One host call per context at a time.
 *
 * mkf_fit_host / mkf_fit_backward_host: same semantics as mkf_fit / mkf_fit_backward, every pointer (hits arrays
 * included; hits->rec is ignored) in host memory. The hits go first; the tracks then travel in ranges of 256 k on three
 * streams (copy in, fit, copy out) so that copies and kernels overlap. h2d_bytes/d2h_bytes (may be NULL) receive the
 * bytes copied each way. */
int mkf_fit_host(mkf_ctx*, const mkf_hits* hits_host, const mkf_states* seeds_host, const signed char* plan,
            const int* track_hits, int max_plan_len, mkf_states* out_host, float* chi2, int* nfit, unsigned* status,
            long long* h2d_bytes, long long* d2h_bytes);
int mkf_fit_backward_host(mkf_ctx*, const mkf_hits* hits_host, const mkf_states* seeds_host, const signed char* plan,
            const int* track_hits, int max_plan_len, mkf_states* out_host, float* chi2, int* nfit, unsigned* status,
            long long* h2d_bytes, long long* d2h_bytes);
/* mkf_build_hit_index + mkf_build_tracks (+ mkf_remove_duplicates if keep != NULL; seeds must then be grouped
 * by event in ascending order) on host buffers. */
int mkf_build_host(mkf_ctx*, const mkf_hits* hits_host, const mkf_states* seeds_host, const int* seed_event,
            const int* seed_hits, const signed char* plan, int max_plan_len, mkf_states* out_host, float* chi2,
            float* score, int* nhits, int* nmiss, int* hit_ids, unsigned* status, unsigned char* keep,
            long long* h2d_bytes, long long* d2h_bytes);
/* mkf_cluster_strips on host buffers (pinned memory makes the copies asynchronous). Device memory comes from the
 * context's arena, so repeated calls pay no allocation ("using a memory pool to pay the allocation
 * overhead only at the beginning and end of job"). *out->n_clusters is the number found; the records are copied
 * only if they all fit (n_clusters <= capacity), see mkf_cluster_strips. */
int mkf_cluster_strips_host(mkf_ctx*, const mkf_strips* strips_host, const mkf_strip_params*, const mkf_clusters* out_host,
            long long* h2d_bytes, long long* d2h_bytes);
#ifdef __cplusplus
}
#endif
#endif
