// mkf_host.cu — workspace sizing and the host-buffer entry points (end-to-end use: H2D copy, kernels, D2H copy).
//
// PAPER.md:69 found host<->device transfers and allocations to be > 90 % of the GPU time of single events and names the
// remedies: "processing multiple events concurrently, thus allowing for asynchronous memory transfer, and ... a memory
// pool to pay the allocation overhead only at the beginning and end of job". Here: the context owns a grow-only device
// arena, three streams and an event pool (mkf_host_state), so a repeated call allocates nothing; mkf_fit_host works on
// ranges of tracks, each range copied in on one stream, fitted on a second and copied out on a third, so that the
// copies of one range overlap the kernel and the copies of its neighbours.
#include "mkf_ctx.h"
#include <vector>

namespace mkf {
size_t hit_index_ws_bytes(const mkf_ctx* c, int n_events, int n_hits);
size_t dedup_ws_bytes(int n_hits, int n, int mpl);
size_t strips_ws_bytes(int n_strips, int capacity);
size_t build_ws_bytes(const mkf_ctx* c, int n_events, int n_seeds);
size_t smooth_ws_bytes(int n, int mpl);
int fit_launch(mkf_ctx* c, bool backward, const FitArgs& a, cudaStream_t st);
}
using namespace mkf;

extern "C" size_t mkf_workspace_bytes(const mkf_ctx* c, int call_id, int n_events, int n_hits, int n_seeds) {
  if (!c || n_events < 0 || n_hits < 0 || n_seeds < 0) return 0;
  switch (call_id) {
    case MKF_CALL_BUILD_HIT_INDEX: return hit_index_ws_bytes(c, n_events, n_hits);
    case MKF_CALL_REMOVE_DUPLICATES: return dedup_ws_bytes(n_hits, n_seeds, c->max_plan_len);
    case MKF_CALL_CLUSTER_STRIPS: return strips_ws_bytes(n_hits, n_seeds);
    case MKF_CALL_BUILD_TRACKS: return build_ws_bytes(c, n_events, n_seeds);
    case MKF_CALL_FIT_SMOOTH: return smooth_ws_bytes(n_seeds, c->max_plan_len);
    case MKF_CALL_BUILD_TRACKS_OVERLAP: return build_ws_bytes(c, n_events, n_seeds) + align256((size_t)n_seeds * c->max_plan_len * 8 * 4);
    default: return 0;      // the fit keeps everything in registers
  }
}

namespace mkf {
void host_state_free(mkf_ctx* c) {
  mkf_host_state* h = c->host;
  if (!h) return;
  if (h->s_in) { cudaStreamSynchronize(h->s_in); cudaStreamSynchronize(h->s_k); cudaStreamSynchronize(h->s_out); }
  for (int k = 0; k < h->n_ev; k++) cudaEventDestroy(h->ev[k]);
  if (h->s_in) { cudaStreamDestroy(h->s_in); cudaStreamDestroy(h->s_k); cudaStreamDestroy(h->s_out); }
  if (h->base) cudaFree(h->base);
  delete h;
  c->host = nullptr;
}
}  // namespace mkf

namespace {
constexpr int FIT_CHUNK = 256 * 1024;        // tracks per range of mkf_fit_host (a multiple of the fit CTA)
constexpr int MAX_EV = 128;

// Bump allocator over the context's arena for the duration of one host call.
struct Arena {
  mkf_host_state* h; size_t used = 0; cudaError_t err = cudaSuccess; long long h2d = 0, d2h = 0; int ev_used = 0;
  // need: upper bound of the bytes this call takes from the arena
  Arena(mkf_ctx* c, size_t need) {
    if (!c->host) c->host = new mkf_host_state();
    h = c->host;
    if (!h->s_in) {
      err = cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking);
      if (err == cudaSuccess) err = cudaStreamCreateWithFlags(&h->s_k, cudaStreamNonBlocking);
      if (err == cudaSuccess) err = cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking);
    }
    if (err == cudaSuccess && h->cap < need) {                  // grow: the only allocation a host call ever makes
      if (h->base) { cudaDeviceSynchronize(); cudaFree(h->base); h->base = nullptr; h->cap = 0; }
      const size_t want = need + need / 8;
      err = cudaMalloc((void**)&h->base, want);
      if (err == cudaSuccess) h->cap = want;
    }
  }
  static size_t pad(size_t b) { return (b + 255) & ~(size_t)255; }
  template <class T> T* alloc(size_t count) {
    const size_t b = pad(count * sizeof(T));
    if (err != cudaSuccess) return nullptr;
    if (used + b > h->cap) { err = cudaErrorMemoryAllocation; return nullptr; }
    T* p = (T*)(h->base + used); used += b; return p;
  }
  template <class T> T* up(const T* host, size_t count, cudaStream_t st) {
    T* d = alloc<T>(count);
    if (err == cudaSuccess && count) { err = cudaMemcpyAsync(d, host, count * sizeof(T), cudaMemcpyHostToDevice, st); h2d += (long long)(count * sizeof(T)); }
    return d;
  }
  template <class T> void down(T* host, const T* dev, size_t count, cudaStream_t st) {
    if (err == cudaSuccess && count) { err = cudaMemcpyAsync(host, dev, count * sizeof(T), cudaMemcpyDeviceToHost, st); d2h += (long long)(count * sizeof(T)); }
  }
  // columns [c0, c0 + cnt) of a [rows][ld] plane-major array: one strided copy
  template <class T> void up_cols(T* dev, const T* host, size_t ld, size_t rows, size_t c0, size_t cnt, cudaStream_t st) {
    if (err == cudaSuccess && cnt) {
      err = cudaMemcpy2DAsync(dev + c0, ld * sizeof(T), host + c0, ld * sizeof(T), cnt * sizeof(T), rows, cudaMemcpyHostToDevice, st);
      h2d += (long long)(rows * cnt * sizeof(T));
    }
  }
  template <class T> void down_cols(T* host, const T* dev, size_t ld, size_t rows, size_t c0, size_t cnt, cudaStream_t st) {
    if (err == cudaSuccess && cnt) {
      err = cudaMemcpy2DAsync(host + c0, ld * sizeof(T), dev + c0, ld * sizeof(T), cnt * sizeof(T), rows, cudaMemcpyDeviceToHost, st);
      d2h += (long long)(rows * cnt * sizeof(T));
    }
  }
  // `to` waits for everything enqueued on `from` so far
  void chain(cudaStream_t from, cudaStream_t to) {
    if (err != cudaSuccess) return;
    if (ev_used == MAX_EV) { err = cudaStreamSynchronize(from); return; }
    if (ev_used == h->n_ev) { err = cudaEventCreateWithFlags(&h->ev[h->n_ev], cudaEventDisableTiming); if (err != cudaSuccess) return; h->n_ev++; }
    cudaEvent_t e = h->ev[ev_used++];
    err = cudaEventRecord(e, from);
    if (err == cudaSuccess) err = cudaStreamWaitEvent(to, e, 0);
  }
  void finish() {
    if (err == cudaSuccess) err = cudaStreamSynchronize(h->s_in);
    if (err == cudaSuccess) err = cudaStreamSynchronize(h->s_k);
    if (err == cudaSuccess) err = cudaStreamSynchronize(h->s_out);
  }
};

size_t hits_bytes(const mkf_ctx* c, const mkf_hits* h) {
  return Arena::pad((size_t)h->n_events * (c->g.n_layers + 1) * 4) + 3 * Arena::pad((size_t)h->n_hits * 4) + Arena::pad((size_t)h->n_hits * 24);
}
mkf_hits upload_hits(Arena& A, const mkf_ctx* c, const mkf_hits* h, cudaStream_t st) {
  mkf_hits d = *h;
  const size_t nh = (size_t)h->n_hits;
  d.layer_off = A.up(h->layer_off, (size_t)h->n_events * (c->g.n_layers + 1), st);
  d.x = A.up(h->x, nh, st); d.y = A.up(h->y, nh, st); d.z = A.up(h->z, nh, st); d.V = A.up(h->V, 6 * nh, st);
  d.rec = nullptr; d.module = nullptr;
  return d;
}

int fit_host(mkf_ctx* c, bool backward, const mkf_hits* h, const mkf_states* seeds, const signed char* plan,
             const int* track_hits, int max_plan_len, mkf_states* out, float* chi2, int* nfit,
             unsigned* status, long long* h2d_bytes, long long* d2h_bytes) {
  if (!c) return MKF_INVALID_ARG;
  if (!h || !seeds || !out || !plan || !track_hits || !chi2 || !nfit || !status || seeds->n < 0 || out->n != seeds->n || max_plan_len < 1)
    return fail(c, MKF_INVALID_ARG, "mkf_fit_host: bad argument");
  const size_t n = (size_t)seeds->n, mpl = (size_t)max_plan_len;
  const size_t need = hits_bytes(c, h) + Arena::pad(n * 24) * 2 + Arena::pad(n * 84) * 2 + 2 * Arena::pad(n) + Arena::pad(n * mpl * 4) +
                      3 * Arena::pad(n * 4) + 4096;
  Arena A(c, need);
  cudaStream_t s_in = A.h->s_in, s_k = A.h->s_k, s_out = A.h->s_out;
  // the hits first (track_hits may name any of them), then the tracks range by range
  mkf_hits dh = upload_hits(A, c, h, s_in);
  float* dpar = A.alloc<float>(6 * n); float* dcov = A.alloc<float>(21 * n); signed char* dq = A.alloc<signed char>(n);
  signed char* dplan = A.alloc<signed char>(n); int* dth = A.alloc<int>(n * mpl);
  float* opar = A.alloc<float>(6 * n); float* ocov = A.alloc<float>(21 * n);
  float* dchi2 = A.alloc<float>(n); int* dnfit = A.alloc<int>(n); unsigned* dstat = A.alloc<unsigned>(n);
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_fit_host: staging");
  for (size_t c0 = 0; c0 < n; c0 += FIT_CHUNK) {
    const size_t cnt = n - c0 < (size_t)FIT_CHUNK ? n - c0 : (size_t)FIT_CHUNK;
    A.up_cols(dpar, seeds->par, n, 6, c0, cnt, s_in); A.up_cols(dcov, seeds->cov, n, 21, c0, cnt, s_in);
    A.up_cols(dq, seeds->q, n, 1, c0, cnt, s_in); A.up_cols(dplan, plan, n, 1, c0, cnt, s_in);
    A.up_cols(dth, track_hits, n, mpl, c0, cnt, s_in);
    A.chain(s_in, s_k);
    if (A.err != cudaSuccess) break;
    FitArgs a;
    a.hits = hits_dev(&dh);
    a.n = (int)cnt; a.ld = (int)n; a.par = dpar + c0; a.cov = dcov + c0; a.q = dq + c0; a.plan = dplan + c0;
    a.track_hits = dth + c0; a.max_plan_len = max_plan_len;
    a.par_out = opar + c0; a.cov_out = ocov + c0; a.chi2 = dchi2 + c0; a.nfit = dnfit + c0; a.status = dstat + c0;
    const int rc = fit_launch(c, backward, a, s_k);
    if (rc) { A.finish(); return rc; }
    A.chain(s_k, s_out);
    A.down_cols(out->par, opar, n, 6, c0, cnt, s_out); A.down_cols(out->cov, ocov, n, 21, c0, cnt, s_out);
    A.down_cols(chi2, dchi2, n, 1, c0, cnt, s_out); A.down_cols(nfit, dnfit, n, 1, c0, cnt, s_out);
    A.down_cols(status, dstat, n, 1, c0, cnt, s_out);
  }
  A.finish();
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_fit_host");
  if (h2d_bytes) *h2d_bytes = A.h2d;
  if (d2h_bytes) *d2h_bytes = A.d2h;
  return MKF_OK;
}
}  // namespace

extern "C" int mkf_fit_host(mkf_ctx* c, const mkf_hits* h, const mkf_states* seeds, const signed char* plan,
                            const int* track_hits, int max_plan_len, mkf_states* out, float* chi2, int* nfit,
                            unsigned* status, long long* h2d_bytes, long long* d2h_bytes) {
  return fit_host(c, false, h, seeds, plan, track_hits, max_plan_len, out, chi2, nfit, status, h2d_bytes, d2h_bytes);
}
extern "C" int mkf_fit_backward_host(mkf_ctx* c, const mkf_hits* h, const mkf_states* seeds, const signed char* plan,
                            const int* track_hits, int max_plan_len, mkf_states* out, float* chi2, int* nfit,
                            unsigned* status, long long* h2d_bytes, long long* d2h_bytes) {
  return fit_host(c, true, h, seeds, plan, track_hits, max_plan_len, out, chi2, nfit, status, h2d_bytes, d2h_bytes);
}

extern "C" int mkf_build_host(mkf_ctx* c, const mkf_hits* h, const mkf_states* seeds, const int* seed_event,
                              const int* seed_hits, const signed char* plan, int max_plan_len, mkf_states* out,
                              float* chi2, float* score, int* nhits, int* nmiss, int* hit_ids, unsigned* status,
                              unsigned char* keep, long long* h2d_bytes, long long* d2h_bytes) {
  if (!c) return MKF_INVALID_ARG;
  if (!h || !seeds || !out || !seed_event || !seed_hits || !plan || !chi2 || !score || !nhits || !nmiss || !hit_ids || !status ||
      seeds->n < 0 || out->n != seeds->n || max_plan_len < 1 || h->n_events < 1)
    return fail(c, MKF_INVALID_ARG, "mkf_build_host: bad argument");
  const size_t n = (size_t)seeds->n, nh = (size_t)h->n_hits, mpl = (size_t)max_plan_len;
  const int nev = h->n_events;
  std::vector<int> toff;
  if (keep) {                                                  // track_off from seed_event (seeds grouped by event, ascending)
    toff.assign((size_t)nev + 1, 0);
    for (size_t i = 0; i < n; i++) {
      const int e = seed_event[i];
      if (e < 0 || e >= nev || (i > 0 && e < seed_event[i - 1])) return fail(c, MKF_INVALID_ARG, "mkf_build_host: seeds not grouped by event");
      toff[(size_t)e + 1]++;
    }
    for (int e = 0; e < nev; e++) toff[(size_t)e + 1] += toff[(size_t)e];
  }
  const size_t nbins = (size_t)nev * c->g.n_layers * c->g.n_phi * c->g.n_eta;
  const size_t ws1 = mkf_workspace_bytes(c, MKF_CALL_BUILD_HIT_INDEX, nev, h->n_hits, seeds->n);
  const size_t ws2 = keep ? mkf_workspace_bytes(c, MKF_CALL_REMOVE_DUPLICATES, nev, h->n_hits, seeds->n) : 0;
  const size_t ws3 = mkf_workspace_bytes(c, MKF_CALL_BUILD_TRACKS, nev, h->n_hits, seeds->n);
  const size_t wsb = (ws1 > ws2 ? ws1 : ws2) > ws3 ? (ws1 > ws2 ? ws1 : ws2) : ws3;
  const size_t need = hits_bytes(c, h) + Arena::pad(n * 24) * 2 + Arena::pad(n * 84) * 2 + 3 * Arena::pad(n) + Arena::pad(n * 4) * 7 +
                      Arena::pad(n * 12) + Arena::pad(n * mpl * 4) + Arena::pad((nbins + 1) * 4) + Arena::pad(nh * 4) +
                      Arena::pad((size_t)nev * c->g.n_layers * 8) + Arena::pad(nh * 48 + 16) + Arena::pad(wsb) + Arena::pad(((size_t)nev + 1) * 4) * 2 + 8192;
  Arena A(c, need);
  cudaStream_t s_in = A.h->s_in, s_k = A.h->s_k, s_out = A.h->s_out;
  mkf_hits dh = upload_hits(A, c, h, s_in);
  A.chain(s_in, s_k);                                          // the hit index starts while the seeds are still on their way
  mkf_hit_index idx;
  idx.bin_off = A.alloc<unsigned>(nbins + 1); idx.sorted_id = A.alloc<int>(nh); idx.vmax = A.alloc<float>((size_t)nev * c->g.n_layers * 2);
  idx.packed = A.alloc<float>(12 * nh + 4);
  char* ws = A.alloc<char>(wsb);
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_build_host: staging");
  int rc = mkf_build_hit_index(c, &dh, &idx, ws, wsb, s_k);
  if (rc) { A.finish(); return rc; }
  mkf_states ds, dout;
  ds.n = dout.n = seeds->n;
  ds.par = A.up(seeds->par, 6 * n, s_in); ds.cov = A.up(seeds->cov, 21 * n, s_in); ds.q = A.up(seeds->q, n, s_in);
  const signed char* dplan = A.up(plan, n, s_in);
  const int* dev_ev = A.up(seed_event, n, s_in);
  const int* dsh = A.up(seed_hits, 3 * n, s_in);
  const int* dtoff = keep ? A.up(toff.data(), toff.size(), s_in) : nullptr;
  A.chain(s_in, s_k);
  dout.par = A.alloc<float>(6 * n); dout.cov = A.alloc<float>(21 * n); dout.q = ds.q;
  float* dchi2 = A.alloc<float>(n); float* dscore = A.alloc<float>(n);
  int* dnh = A.alloc<int>(n); int* dnm = A.alloc<int>(n); int* dhid = A.alloc<int>(n * mpl);
  unsigned* dstat = A.alloc<unsigned>(n);
  unsigned char* dkeep = keep ? A.alloc<unsigned char>(n) : nullptr; int* dnk = keep ? A.alloc<int>((size_t)nev) : nullptr;
  if (A.err != cudaSuccess) { A.finish(); return cuda_fail(c, A.err, "mkf_build_host: staging"); }
  rc = mkf_build_tracks(c, &dh, &idx, &ds, dev_ev, dsh, dplan, max_plan_len, &dout, dchi2, dscore, dnh, dnm, dhid, dstat, ws, wsb, s_k);
  if (rc) { A.finish(); return rc; }
  A.chain(s_k, s_out);                                         // the tracks go home while the duplicates are being removed
  A.down(out->par, dout.par, 6 * n, s_out); A.down(out->cov, dout.cov, 21 * n, s_out);
  A.down(chi2, dchi2, n, s_out); A.down(score, dscore, n, s_out); A.down(nhits, dnh, n, s_out); A.down(nmiss, dnm, n, s_out);
  A.down(hit_ids, dhid, n * mpl, s_out); A.down(status, dstat, n, s_out);
  if (keep) {
    rc = mkf_remove_duplicates(c, nev, seeds->n, h->n_hits, dtoff, dhid, max_plan_len, dnh, dscore, dkeep, dnk, ws, wsb, s_k);
    if (rc) { A.finish(); return rc; }
    A.down(keep, dkeep, n, s_k);
  }
  A.finish();                                                  // also keeps `toff` alive until its copy is done
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_build_host");
  if (h2d_bytes) *h2d_bytes = A.h2d;
  if (d2h_bytes) *d2h_bytes = A.d2h;
  return MKF_OK;
}

extern "C" int mkf_cluster_strips_host(mkf_ctx* c, const mkf_strips* s, const mkf_strip_params* p, const mkf_clusters* out,
                                       long long* h2d_bytes, long long* d2h_bytes) {
  if (!c) return MKF_INVALID_ARG;
  if (!s || !p || !out || s->n_strips < 0 || s->n_modules < 0 || out->capacity < 0 || !out->n_clusters ||
      (s->n_strips > 0 && (!s->module_off || !s->adc || !s->noise || !s->bad)))
    return fail(c, MKF_INVALID_ARG, "mkf_cluster_strips_host: bad argument");
  const size_t n = (size_t)s->n_strips, cap = (size_t)out->capacity;
  const size_t wsb = strips_ws_bytes(s->n_strips, out->capacity);
  const size_t need = Arena::pad(((size_t)s->n_modules + 1) * 4) + Arena::pad(n * 2) + Arena::pad(n * 4) + Arena::pad(n) + 5 * Arena::pad(cap * 4) +
                      Arena::pad(wsb) + 4096;
  Arena A(c, need);
  cudaStream_t st = A.h->s_k;
  mkf_strips ds = *s;
  ds.module_off = A.up(s->module_off, (size_t)s->n_modules + 1, st);
  ds.adc = A.up(s->adc, n, st); ds.noise = A.up(s->noise, n, st); ds.bad = A.up(s->bad, n, st);
  mkf_clusters dc = *out;
  dc.module = A.alloc<int>(cap); dc.first = A.alloc<int>(cap); dc.last = A.alloc<int>(cap);
  dc.charge = A.alloc<unsigned>(cap); dc.bary = A.alloc<float>(cap); dc.n_clusters = A.alloc<int>(1);
  char* ws = A.alloc<char>(wsb);
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_cluster_strips_host: staging");
  const int rc = mkf_cluster_strips(c, &ds, p, &dc, ws, wsb, st);
  if (rc) { A.finish(); return rc; }
  A.down(out->n_clusters, dc.n_clusters, 1, st);
  if (A.err == cudaSuccess) A.err = cudaStreamSynchronize(st);             // the count decides how much comes back
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_cluster_strips_host");
  const size_t k = *out->n_clusters <= out->capacity ? (size_t)*out->n_clusters : 0;      // overflow: only the count is defined
  A.down(out->module, dc.module, k, st); A.down(out->first, dc.first, k, st); A.down(out->last, dc.last, k, st);
  A.down(out->charge, dc.charge, k, st); A.down(out->bary, dc.bary, k, st);
  A.finish();
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_cluster_strips_host");
  if (h2d_bytes) *h2d_bytes = A.h2d;
  if (d2h_bytes) *d2h_bytes = A.d2h;
  return MKF_OK;
}
