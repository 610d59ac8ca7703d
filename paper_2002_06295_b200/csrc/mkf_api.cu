// mkf_api.cu — context management and the fit entry point of libmkf.so (see include/mkf.h).
#include "mkf_ctx.h"

using namespace mkf;

extern "C" int mkf_create(mkf_ctx** out, const mkf_geometry* geom, const mkf_params* prm) {
  if (!out || !geom || !prm || !geom->layers || !geom->plan_off || !geom->plan_layers) return MKF_INVALID_ARG;
  if (geom->n_layers < 1 || geom->n_plans < 1 || geom->n_phi_bins < 1 || geom->n_eta_bins < 1) return MKF_INVALID_ARG;
  if (geom->n_layers > MAX_LAYERS || geom->n_plans > MAX_PLANS) return MKF_UNSUPPORTED;
  if (geom->plan_off[0] != 0 || geom->plan_off[geom->n_plans] > MAX_PLAN_STEPS) return MKF_UNSUPPORTED;
  if (prm->max_cand < 1 || prm->max_cand > MAX_CAND) return MKF_UNSUPPORTED;
  mkf_ctx* c = new mkf_ctx();
  memset(c, 0, sizeof(*c));
  c->g.n_layers = geom->n_layers; c->g.n_plans = geom->n_plans;
  c->g.n_phi = geom->n_phi_bins; c->g.n_eta = geom->n_eta_bins; c->g.bz = geom->bz;
  for (int l = 0; l < geom->n_layers; l++) {
    const mkf_layer& s = geom->layers[l];
    LayerDev& d = c->g.layers[l];
    d.kind = s.kind; d.pos = s.pos; d.lo = s.lo; d.hi = s.hi; d.xx0 = s.xx0; d.eta_lo = s.eta_lo; d.eta_hi = s.eta_hi;
    c->g.bz_layer[l] = geom->bz_layer ? geom->bz_layer[l] : geom->bz;
    if ((s.kind != 0 && s.kind != 1) || !(s.eta_hi > s.eta_lo) || (s.kind == 0 && !(s.pos > 0.f))) { delete c; return MKF_INVALID_ARG; }
  }
  int mpl = 0;
  for (int p = 0; p <= geom->n_plans; p++) c->g.plan_off[p] = geom->plan_off[p];
  for (int p = 0; p < geom->n_plans; p++) {
    const int len = geom->plan_off[p + 1] - geom->plan_off[p];
    if (len < 0) { delete c; return MKF_INVALID_ARG; }
    if (len > mpl) mpl = len;
  }
  for (int k = 0; k < geom->plan_off[geom->n_plans]; k++) {
    const int l = geom->plan_layers[k];
    if (l < 0 || l >= geom->n_layers) { delete c; return MKF_INVALID_ARG; }
    c->g.plan_layers[k] = (unsigned char)l;
  }
  c->max_plan_len = mpl;
  c->p.chi2_cut = prm->chi2_cut; c->p.max_cand = prm->max_cand; c->p.max_consec_miss = prm->max_consec_miss;
  c->p.min_hits_keep = prm->min_hits_keep; c->p.score_hit = prm->score_hit; c->p.score_miss = prm->score_miss;
  c->p.graze_cos_min = prm->graze_cos_min; c->p.material_flags = prm->material_flags; c->p.dup_frac = prm->dup_frac;
  *out = c;
  return MKF_OK;
}

namespace mkf { void host_state_free(mkf_ctx*); }
extern "C" void mkf_destroy(mkf_ctx* c) { if (c) host_state_free(c); delete c; }
extern "C" const char* mkf_last_error(const mkf_ctx* c) { return c ? c->err : "null context"; }
extern "C" long long mkf_launch_count(const mkf_ctx* c) { return c ? c->launches : 0; }
extern "C" int mkf_max_plan_len(const mkf_ctx* c) { return c ? c->max_plan_len : 0; }
extern "C" int mkf_set_build_counters(mkf_ctx* c, unsigned long long* counters) { if (!c) return MKF_INVALID_ARG; c->build_counters = counters; return MKF_OK; }

// ---- 48-byte hit records (mkf_hits.rec): one streaming pass over the SoA planes ------------------------------
__global__ void __launch_bounds__(256) mkf_pack_hits_kernel(int n, const float* __restrict__ x, const float* __restrict__ y,
                                                            const float* __restrict__ z, const float* __restrict__ V, float4* __restrict__ rec) {
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i >= n) return;
  const size_t nh = (size_t)n;
  float4* r = rec + (size_t)3 * i;
  r[0] = make_float4(x[i], y[i], z[i], V[i]);
  r[1] = make_float4(V[nh + i], V[2 * nh + i], V[3 * nh + i], V[4 * nh + i]);
  r[2] = make_float4(V[5 * nh + i], 0.f, 0.f, 0.f);
}

extern "C" int mkf_pack_hits(mkf_ctx* c, const mkf_hits* h, float* rec_out, void* stream) {
  if (!c) return MKF_INVALID_ARG;
  if (!h || h->n_hits < 0) return fail(c, MKF_INVALID_ARG, "mkf_pack_hits: bad argument");
  if (h->n_hits == 0) return MKF_OK;
  if (!h->x || !h->y || !h->z || !h->V || !rec_out || ((size_t)rec_out & 15)) return fail(c, MKF_INVALID_ARG, "mkf_pack_hits: null or misaligned array");
  mkf_pack_hits_kernel<<<(h->n_hits + 255) / 256, 256, 0, (cudaStream_t)stream>>>(h->n_hits, h->x, h->y, h->z, h->V, (float4*)rec_out);
  MKF_LAUNCHED(c, "mkf_pack_hits_kernel");
  return MKF_OK;
}

// ---- fit (a11 / C7): one thread per track, state and covariance in registers for the whole layer loop ----
#ifndef MKF_FIT_BLOCK
#define MKF_FIT_BLOCK 128
#endif
constexpr int FIT_BLOCK = MKF_FIT_BLOCK;
#ifndef MKF_FIT_MIN_BLOCKS
#define MKF_FIT_MIN_BLOCKS 5
#endif

template <bool STRAG, bool PLANES>
__global__ void __launch_bounds__(FIT_BLOCK, MKF_FIT_MIN_BLOCKS) mkf_fit_kernel(const __grid_constant__ GeomDev g,
                                                            const __grid_constant__ ParamsDev p,
                                                            const __grid_constant__ FitArgs a) {
  const int i = blockIdx.x * FIT_BLOCK + threadIdx.x;
  if (i < a.n) fit_one<STRAG, PLANES>(g, p, a, i);
}

template <bool STRAG, bool PLANES>
__global__ void __launch_bounds__(FIT_BLOCK, MKF_FIT_MIN_BLOCKS) mkf_fit_backward_kernel(const __grid_constant__ GeomDev g,
                                                                        const __grid_constant__ ParamsDev p,
                                                                        const __grid_constant__ FitArgs a) {
  const int i = blockIdx.x * FIT_BLOCK + threadIdx.x;
  if (i < a.n) fit_one_backward<STRAG, PLANES>(g, p, a, i);
}

static int fit_common(mkf_ctx* c, bool backward, const mkf_hits* h, const mkf_states* seeds, const signed char* plan,
                      const int* track_hits, int max_plan_len, mkf_states* out, float* chi2, int* nfit, unsigned* status,
                      void* stream);

extern "C" int mkf_fit_backward(mkf_ctx* c, const mkf_hits* h, const mkf_states* seeds, const signed char* plan,
                                const int* track_hits, int max_plan_len, mkf_states* out, float* chi2, int* nfit,
                                unsigned* status, void* ws, size_t ws_bytes, void* stream) {
  (void)ws; (void)ws_bytes;
  return fit_common(c, true, h, seeds, plan, track_hits, max_plan_len, out, chi2, nfit, status, stream);
}

extern "C" int mkf_fit(mkf_ctx* c, const mkf_hits* h, const mkf_states* seeds, const signed char* plan,
                       const int* track_hits, int max_plan_len, mkf_states* out, float* chi2, int* nfit,
                       unsigned* status, void* ws, size_t ws_bytes, void* stream) {
  (void)ws; (void)ws_bytes;
  return fit_common(c, false, h, seeds, plan, track_hits, max_plan_len, out, chi2, nfit, status, stream);
}

namespace mkf {
// One launch over the tracks [0, a.n) of FitArgs (plane stride a.ld); used by mkf_fit / mkf_fit_backward and, on
// track ranges, by the host-buffer entry points.
int fit_launch(mkf_ctx* c, bool backward, const FitArgs& a, cudaStream_t st) {
  if (a.n <= 0) return MKF_OK;
  const int grid = (a.n + FIT_BLOCK - 1) / FIT_BLOCK;
  const bool strag = (c->p.material_flags & 4) != 0;        // R12: its code is only in the kernels that need it
  const bool pl = a.hits.rec == nullptr;                    // hits as planes: instances without the per-hit test of the record pointer
  void (*kern)(GeomDev, ParamsDev, FitArgs) =
      backward ? (strag ? (pl ? mkf_fit_backward_kernel<true, true> : mkf_fit_backward_kernel<true, false>)
                        : (pl ? mkf_fit_backward_kernel<false, true> : mkf_fit_backward_kernel<false, false>))
               : (strag ? (pl ? mkf_fit_kernel<true, true> : mkf_fit_kernel<true, false>)
                        : (pl ? mkf_fit_kernel<false, true> : mkf_fit_kernel<false, false>));
  kern<<<grid, FIT_BLOCK, 0, st>>>(c->g, c->p, a);
  MKF_LAUNCHED(c, backward ? "mkf_fit_backward_kernel" : "mkf_fit_kernel");
  return MKF_OK;
}
}  // namespace mkf

static int fit_common(mkf_ctx* c, bool backward, const mkf_hits* h, const mkf_states* seeds, const signed char* plan,
                      const int* track_hits, int max_plan_len, mkf_states* out, float* chi2, int* nfit, unsigned* status,
                      void* stream) {
  if (!c) return MKF_INVALID_ARG;
  if (!h || !seeds || !out) return fail(c, MKF_INVALID_ARG, "mkf_fit: null argument");
  if (seeds->n < 0 || out->n != seeds->n || max_plan_len < 1) return fail(c, MKF_INVALID_ARG, "mkf_fit: bad sizes");
  if (seeds->n == 0) return MKF_OK;                      // nothing to do; array pointers may be null
  if (!plan || !track_hits || !chi2 || !nfit || !status) return fail(c, MKF_INVALID_ARG, "mkf_fit: null argument");
  if (!h->x || !h->y || !h->z || !h->V || !seeds->par || !seeds->cov || !seeds->q || !out->par || !out->cov)
    return fail(c, MKF_INVALID_ARG, "mkf_fit: null array");
  if ((size_t)h->rec & 15) return fail(c, MKF_INVALID_ARG, "mkf_fit: hit records not 16-byte aligned");
  FitArgs a;
  a.hits = hits_dev(h);
  a.n = seeds->n; a.ld = seeds->n; a.par = seeds->par; a.cov = seeds->cov; a.q = seeds->q; a.plan = plan;
  a.track_hits = track_hits; a.max_plan_len = max_plan_len;
  a.par_out = out->par; a.cov_out = out->cov; a.chi2 = chi2; a.nfit = nfit; a.status = status;
  return fit_launch(c, backward, a, (cudaStream_t)stream);
}

// ---- two-filter smoother (reading R14) ----------------------------------------------------------------
#ifndef MKF_SMOOTH_MIN_BLOCKS
#define MKF_SMOOTH_MIN_BLOCKS 3
#endif
__global__ void __launch_bounds__(FIT_BLOCK, MKF_SMOOTH_MIN_BLOCKS) mkf_fit_smooth_kernel(const __grid_constant__ GeomDev g, const __grid_constant__ ParamsDev p,
                                                                   const __grid_constant__ SmoothArgs a) {
  const int i = blockIdx.x * FIT_BLOCK + threadIdx.x;
  if (i < a.f.n) fit_smooth_one(g, p, a, i);
}

namespace mkf { size_t smooth_ws_bytes(int n, int mpl) { return align256((size_t)SM_NF * mpl * n * sizeof(float)); } }

extern "C" int mkf_fit_smooth(mkf_ctx* c, const mkf_hits* h, const mkf_states* seeds, const signed char* plan, const int* track_hits,
                              int max_plan_len, float* par_s, float* cov_s, float* chi2, int* nfit, unsigned* status,
                              void* ws, size_t ws_bytes, void* stream) {
  if (!c) return MKF_INVALID_ARG;
  if (!h || !seeds) return fail(c, MKF_INVALID_ARG, "mkf_fit_smooth: null argument");
  if (seeds->n < 0 || max_plan_len < 1) return fail(c, MKF_INVALID_ARG, "mkf_fit_smooth: bad sizes");
  if (seeds->n == 0) return MKF_OK;
  if (!plan || !track_hits || !par_s || !cov_s || !chi2 || !nfit || !status || !h->x || !h->y || !h->z || !h->V ||
      !seeds->par || !seeds->cov || !seeds->q)
    return fail(c, MKF_INVALID_ARG, "mkf_fit_smooth: null array");
  if ((size_t)h->rec & 15) return fail(c, MKF_INVALID_ARG, "mkf_fit_smooth: hit records not 16-byte aligned");
  const size_t need = smooth_ws_bytes(seeds->n, max_plan_len);
  if (ws_bytes < need || !ws) return fail(c, MKF_WORKSPACE_TOO_SMALL, "mkf_fit_smooth: workspace too small");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t n = (size_t)seeds->n;
  cudaError_t e = cudaMemsetAsync(par_s, 0, n * max_plan_len * 6 * sizeof(float), st);
  if (e == cudaSuccess) e = cudaMemsetAsync(cov_s, 0, n * max_plan_len * 21 * sizeof(float), st);
  if (e != cudaSuccess) return cuda_fail(c, e, "mkf_fit_smooth: memset");
  SmoothArgs a;
  a.f.hits = hits_dev(h);
  a.f.n = seeds->n; a.f.ld = seeds->n; a.f.par = seeds->par; a.f.cov = seeds->cov; a.f.q = seeds->q; a.f.plan = plan;
  a.f.track_hits = track_hits; a.f.max_plan_len = max_plan_len;
  a.f.par_out = nullptr; a.f.cov_out = nullptr; a.f.chi2 = chi2; a.f.nfit = nfit; a.f.status = status;
  a.par_s = par_s; a.cov_s = cov_s; a.ws = (float*)ws;
  mkf_fit_smooth_kernel<<<(a.f.n + FIT_BLOCK - 1) / FIT_BLOCK, FIT_BLOCK, 0, st>>>(c->g, c->p, a);
  MKF_LAUNCHED(c, "mkf_fit_smooth_kernel");
  return MKF_OK;
}
