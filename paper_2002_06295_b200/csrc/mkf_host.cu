// mkf_host.cu — workspace sizing and the host-buffer entry points (end-to-end use: H2D copy, kernels, D2H copy).
#include "mkf_ctx.h"
#include <vector>

namespace mkf {
size_t hit_index_ws_bytes(const mkf_ctx* c, int n_events, int n_hits);
size_t dedup_ws_bytes(int n_hits, int n, int mpl);
size_t strips_ws_bytes(int n_strips, int capacity);
}
using namespace mkf;

extern "C" size_t mkf_workspace_bytes(const mkf_ctx* c, int call_id, int n_events, int n_hits, int n_seeds) {
  if (!c || n_events < 0 || n_hits < 0 || n_seeds < 0) return 0;
  switch (call_id) {
    case MKF_CALL_BUILD_HIT_INDEX: return hit_index_ws_bytes(c, n_events, n_hits);
    case MKF_CALL_REMOVE_DUPLICATES: return dedup_ws_bytes(n_hits, n_seeds, c->max_plan_len);
    case MKF_CALL_CLUSTER_STRIPS: return strips_ws_bytes(n_hits, n_seeds);
    default: return 0;      // fit and build keep everything in registers / shared memory
  }
}

namespace {
// Device arena from the stream-ordered pool; everything is released by the destructor.
struct Arena {
  cudaStream_t st = nullptr; std::vector<void*> ptrs; cudaError_t err = cudaSuccess; long long h2d = 0, d2h = 0;
  Arena() { err = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking); }
  ~Arena() { for (void* p : ptrs) cudaFreeAsync(p, st); if (st) { cudaStreamSynchronize(st); cudaStreamDestroy(st); } }
  template <class T> T* alloc(size_t count) {
    void* p = nullptr;
    if (err == cudaSuccess) { err = cudaMallocAsync(&p, count * sizeof(T) + 256, st); if (err == cudaSuccess) ptrs.push_back(p); }
    return (T*)p;
  }
  template <class T> T* up(const T* host, size_t count) {
    T* d = alloc<T>(count);
    if (err == cudaSuccess && count) { err = cudaMemcpyAsync(d, host, count * sizeof(T), cudaMemcpyHostToDevice, st); h2d += (long long)(count * sizeof(T)); }
    return d;
  }
  template <class T> void down(T* host, const T* dev, size_t count) {
    if (err == cudaSuccess && count) { err = cudaMemcpyAsync(host, dev, count * sizeof(T), cudaMemcpyDeviceToHost, st); d2h += (long long)(count * sizeof(T)); }
  }
};

mkf_hits upload_hits(Arena& A, const mkf_ctx* c, const mkf_hits* h) {
  mkf_hits d = *h;
  const size_t nh = (size_t)h->n_hits;
  d.layer_off = A.up(h->layer_off, (size_t)h->n_events * (c->g.n_layers + 1));
  d.x = A.up(h->x, nh); d.y = A.up(h->y, nh); d.z = A.up(h->z, nh); d.V = A.up(h->V, 6 * nh);
  return d;
}
}  // namespace

extern "C" int mkf_fit_host(mkf_ctx* c, const mkf_hits* h, const mkf_states* seeds, const signed char* plan,
                            const int* track_hits, int max_plan_len, mkf_states* out, float* chi2, int* nfit,
                            unsigned* status, long long* h2d_bytes, long long* d2h_bytes) {
  if (!c) return MKF_INVALID_ARG;
  if (!h || !seeds || !out || !plan || !track_hits || !chi2 || !nfit || !status || seeds->n < 0 || out->n != seeds->n || max_plan_len < 1)
    return fail(c, MKF_INVALID_ARG, "mkf_fit_host: bad argument");
  const size_t n = (size_t)seeds->n;
  Arena A;
  mkf_hits dh = upload_hits(A, c, h);
  mkf_states ds, dout;
  ds.n = dout.n = seeds->n;
  ds.par = A.up(seeds->par, 6 * n); ds.cov = A.up(seeds->cov, 21 * n); ds.q = A.up(seeds->q, n);
  const signed char* dplan = A.up(plan, n);
  const int* dth = A.up(track_hits, n * max_plan_len);
  dout.par = A.alloc<float>(6 * n); dout.cov = A.alloc<float>(21 * n); dout.q = ds.q;
  float* dchi2 = A.alloc<float>(n); int* dnfit = A.alloc<int>(n); unsigned* dstat = A.alloc<unsigned>(n);
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_fit_host: staging");
  const int rc = mkf_fit(c, &dh, &ds, dplan, dth, max_plan_len, &dout, dchi2, dnfit, dstat, nullptr, 0, A.st);
  if (rc) return rc;
  A.down(out->par, dout.par, 6 * n); A.down(out->cov, dout.cov, 21 * n);
  A.down(chi2, dchi2, n); A.down(nfit, dnfit, n); A.down(status, dstat, n);
  if (A.err == cudaSuccess) A.err = cudaStreamSynchronize(A.st);
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_fit_host");
  if (h2d_bytes) *h2d_bytes = A.h2d;
  if (d2h_bytes) *d2h_bytes = A.d2h;
  return MKF_OK;
}

extern "C" int mkf_build_host(mkf_ctx* c, const mkf_hits* h, const mkf_states* seeds, const int* seed_event,
                              const int* seed_hits, const signed char* plan, int max_plan_len, mkf_states* out,
                              float* chi2, float* score, int* nhits, int* nmiss, int* hit_ids, unsigned* status,
                              unsigned char* keep, long long* h2d_bytes, long long* d2h_bytes) {
  if (!c) return MKF_INVALID_ARG;
  if (!h || !seeds || !out || !seed_event || !seed_hits || !plan || !chi2 || !score || !nhits || !nmiss || !hit_ids || !status ||
      seeds->n < 0 || out->n != seeds->n || max_plan_len < 1 || h->n_events < 1)
    return fail(c, MKF_INVALID_ARG, "mkf_build_host: bad argument");
  const size_t n = (size_t)seeds->n, nh = (size_t)h->n_hits;
  const int nev = h->n_events;
  Arena A;
  mkf_hits dh = upload_hits(A, c, h);
  mkf_states ds, dout;
  ds.n = dout.n = seeds->n;
  ds.par = A.up(seeds->par, 6 * n); ds.cov = A.up(seeds->cov, 21 * n); ds.q = A.up(seeds->q, n);
  const signed char* dplan = A.up(plan, n);
  const int* dev_ev = A.up(seed_event, n);
  const int* dsh = A.up(seed_hits, 3 * n);
  const size_t nbins = (size_t)nev * c->g.n_layers * c->g.n_phi * c->g.n_eta;
  mkf_hit_index idx;
  idx.bin_off = A.alloc<unsigned>(nbins + 1); idx.sorted_id = A.alloc<int>(nh); idx.vmax = A.alloc<float>((size_t)nev * c->g.n_layers * 2);
  idx.packed = A.alloc<float>(12 * nh);
  const size_t ws1 = mkf_workspace_bytes(c, MKF_CALL_BUILD_HIT_INDEX, nev, h->n_hits, seeds->n);
  const size_t ws2 = keep ? mkf_workspace_bytes(c, MKF_CALL_REMOVE_DUPLICATES, nev, h->n_hits, seeds->n) : 0;
  const size_t wsb = ws1 > ws2 ? ws1 : ws2;
  char* ws = A.alloc<char>(wsb);
  dout.par = A.alloc<float>(6 * n); dout.cov = A.alloc<float>(21 * n); dout.q = ds.q;
  float* dchi2 = A.alloc<float>(n); float* dscore = A.alloc<float>(n);
  int* dnh = A.alloc<int>(n); int* dnm = A.alloc<int>(n); int* dhid = A.alloc<int>(n * max_plan_len);
  unsigned* dstat = A.alloc<unsigned>(n);
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_build_host: staging");
  int rc = mkf_build_hit_index(c, &dh, &idx, ws, wsb, A.st);
  if (rc) return rc;
  rc = mkf_build_tracks(c, &dh, &idx, &ds, dev_ev, dsh, dplan, max_plan_len, &dout, dchi2, dscore, dnh, dnm, dhid, dstat, nullptr, 0, A.st);
  if (rc) return rc;
  if (keep) {
    // track_off from seed_event (seeds grouped by event, ascending)
    std::vector<int> toff((size_t)nev + 1, 0);
    for (size_t i = 0; i < n; i++) {
      const int e = seed_event[i];
      if (e < 0 || e >= nev || (i > 0 && e < seed_event[i - 1])) return fail(c, MKF_INVALID_ARG, "mkf_build_host: seeds not grouped by event");
      toff[(size_t)e + 1]++;
    }
    for (int e = 0; e < nev; e++) toff[(size_t)e + 1] += toff[(size_t)e];
    const int* dtoff = A.up(toff.data(), toff.size());
    unsigned char* dkeep = A.alloc<unsigned char>(n); int* dnk = A.alloc<int>((size_t)nev);
    if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_build_host: staging");
    if (A.err == cudaSuccess) A.err = cudaStreamSynchronize(A.st);      // toff is a local buffer
    rc = mkf_remove_duplicates(c, nev, seeds->n, h->n_hits, dtoff, dhid, max_plan_len, dnh, dscore, dkeep, dnk, ws, wsb, A.st);
    if (rc) return rc;
    A.down(keep, dkeep, n);
  }
  A.down(out->par, dout.par, 6 * n); A.down(out->cov, dout.cov, 21 * n);
  A.down(chi2, dchi2, n); A.down(score, dscore, n); A.down(nhits, dnh, n); A.down(nmiss, dnm, n);
  A.down(hit_ids, dhid, n * max_plan_len); A.down(status, dstat, n);
  if (A.err == cudaSuccess) A.err = cudaStreamSynchronize(A.st);
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
  Arena A;
  mkf_strips ds = *s;
  ds.module_off = A.up(s->module_off, (size_t)s->n_modules + 1);
  ds.adc = A.up(s->adc, n); ds.noise = A.up(s->noise, n); ds.bad = A.up(s->bad, n);
  mkf_clusters dc = *out;
  dc.module = A.alloc<int>(cap); dc.first = A.alloc<int>(cap); dc.last = A.alloc<int>(cap);
  dc.charge = A.alloc<unsigned>(cap); dc.bary = A.alloc<float>(cap); dc.n_clusters = A.alloc<int>(1);
  const size_t wsb = strips_ws_bytes(s->n_strips, out->capacity);
  char* ws = A.alloc<char>(wsb);
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_cluster_strips_host: staging");
  const int rc = mkf_cluster_strips(c, &ds, p, &dc, ws, wsb, A.st);
  if (rc) return rc;
  A.down(out->n_clusters, dc.n_clusters, 1);
  if (A.err == cudaSuccess) A.err = cudaStreamSynchronize(A.st);           // the count decides how much comes back
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_cluster_strips_host");
  const size_t k = (size_t)(*out->n_clusters < out->capacity ? *out->n_clusters : out->capacity);
  A.down(out->module, dc.module, k); A.down(out->first, dc.first, k); A.down(out->last, dc.last, k);
  A.down(out->charge, dc.charge, k); A.down(out->bary, dc.bary, k);
  if (A.err == cudaSuccess) A.err = cudaStreamSynchronize(A.st);
  if (A.err != cudaSuccess) return cuda_fail(c, A.err, "mkf_cluster_strips_host");
  if (h2d_bytes) *h2d_bytes = A.h2d;
  if (d2h_bytes) *d2h_bytes = A.d2h;
  return MKF_OK;
}
