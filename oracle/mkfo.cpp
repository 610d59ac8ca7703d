// mkfo.cpp — the ORACLE: plain float64 CPU restatement of the Kalman-filter hot path (see mkfo.h).
// TEST INFRASTRUCTURE ONLY. Not tuned. Dense 6x6 loops, std::sort, brute-force loops; OpenMP `parallel for`
// over tracks / seeds / events only so that the timed baseline uses the host's cores.
// Citations: PAPER.md:<line> of /root/reference/PAPER.md; C*/U* = readings in DESIGN.md §3.
#include "mkfo.h"
#include <cmath>
#include <cstring>
#include <cstdint>
#include <vector>
#include <algorithm>
#include <limits>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum { IX = 0, IY = 1, IZ = 2, IIPT = 3, IPHI = 4, ITH = 5 };
const double KAPPA = 0.0029979246;      // GeV/(T cm)
const double PI = 3.14159265358979323846;
const double S_BACK = 1e-3;             // cm: largest backward step accepted as "already on the surface" (U5)
const double DISK_GRAZE_COS = 0.05;     // U7 for disks

struct State { double u[6]; double C[36]; int q; };

inline double sinc(double h) { return std::fabs(h) < 1e-8 ? 1.0 - h * h / 6.0 : std::sin(h) / h; }

// C1: exact helix in uniform Bz, transverse path s.
// phi1 = phi0 + w s; x1 = x0 + (sin phi1 - sin phi0)/w; y1 = y0 - (cos phi1 - cos phi0)/w; z1 = z0 + s cot(theta)
// written with sin a - sin b = 2 cos((a+b)/2) sin((a-b)/2) so that w -> 0 is the straight line.
void helix_step(double bz, int q, const double* u, double s, double* u1) {
  double w = -q * KAPPA * bz * u[IIPT];
  double h = 0.5 * w * s;
  u1[IX] = u[IX] + s * sinc(h) * std::cos(u[IPHI] + h);
  u1[IY] = u[IY] + s * sinc(h) * std::sin(u[IPHI] + h);
  u1[IZ] = u[IZ] + s / std::tan(u[ITH]);
  u1[IIPT] = u[IIPT];
  u1[IPHI] = u[IPHI] + w * s;
  u1[ITH] = u[ITH];
}

// C2: transverse path to the cylinder r = R by circle-circle intersection; exit point (outward radial velocity).
// C3: path to the plane z = Z.  Returns false if unreachable (U5, U6).
// dir = +1: forward (outward) step; dir = -1: backward step, s <= 0 (reading R7).
bool path_to_surface(int kind, double pos, double bz, int q, const double* u, double* s_out, int dir = 1) {
  double w = -q * KAPPA * bz * u[IIPT];
  double s;
  if (kind == 1) {
    s = (pos - u[IZ]) * std::tan(u[ITH]);                       // C3
  } else {
    double x0 = u[IX], y0 = u[IY], sp = std::sin(u[IPHI]), cp = std::cos(u[IPHI]);
    double R = pos, r02 = x0 * x0 + y0 * y0;
    if (std::fabs(w) < 1e-14) {                                  // straight line limit
      double A = x0 * cp + y0 * sp, D = R * R - r02, disc = A * A + D;
      if (disc < 0) return false;
      s = -A + std::sqrt(disc);
    } else {
      double cx = x0 - sp / w, cy = y0 + cp / w;                 // centre of the circle
      double B = y0 * cp - x0 * sp;
      double dd = r02 + 2.0 * B / w;                             // d^2 - rho^2 without cancellation
      double d2 = dd + 1.0 / (w * w);
      if (!(d2 > 0)) return false;
      double d = std::sqrt(d2);
      double alpha = (R * R + dd) / (2.0 * d);
      double b2 = R * R - alpha * alpha;
      if (b2 < 0) return false;                                  // circles do not meet
      double beta = std::sqrt(b2);
      double chx = cx / d, chy = cy / d;
      double u0x = sp / w, u0y = -cp / w;                        // P0 - c
      double best_s = 0; double best_vr = -std::numeric_limits<double>::infinity(); bool found = false;
      for (int sg = -1; sg <= 1; sg += 2) {
        double Px = alpha * chx - sg * beta * chy, Py = alpha * chy + sg * beta * chx;
        double dPx = Px - x0, dPy = Py - y0;
        double cross = u0x * dPy - u0y * dPx;
        double dot = 1.0 / (w * w) + u0x * dPx + u0y * dPy;
        double dpsi = std::atan2(cross, dot);                    // turning angle, principal value
        double phi1 = u[IPHI] + dpsi;
        double vr = Px * std::cos(phi1) + Py * std::sin(phi1);   // radial velocity * r
        if (vr > best_vr) { best_vr = vr; best_s = dpsi / w; found = true; }
      }
      if (!found) return false;
      s = best_s;                                                // may be < 0: wrapped principal value
    }
  }
  if (dir > 0 && s < -S_BACK) return false;                      // backward, or forward arc >= pi (U5/U6)
  if (dir < 0 && s > S_BACK) return false;                       // R7: the same rule mirrored
  if (std::fabs(w * s) >= PI) return false;                      // U6
  *s_out = s;
  return true;
}

// C4: F = A + b c^T.
void jacobian(int kind, double pos, double bz, int q, const double* u, const double* u1, double s, double* F) {
  double a = -q * KAPPA * bz, ipt = u[IIPT], w = a * ipt;
  double dx = u1[IX] - u[IX], dy = u1[IY] - u[IY];
  double c1 = std::cos(u1[IPHI]), s1 = std::sin(u1[IPHI]);
  double st = std::sin(u[ITH]), ct = std::cos(u[ITH]);
  double A[36] = {0}; for (int i = 0; i < 6; i++) A[i * 6 + i] = 1.0;
  A[IX * 6 + IPHI] = -dy;
  A[IY * 6 + IPHI] = dx;
  A[IX * 6 + IIPT] = (s * c1 - dx) / ipt;
  A[IY * 6 + IIPT] = (s * s1 - dy) / ipt;
  A[IZ * 6 + ITH] = -s / (st * st);
  A[IPHI * 6 + IIPT] = a * s;
  double b[6] = {c1, s1, ct / st, 0.0, w, 0.0};
  double c[6] = {0, 0, 0, 0, 0, 0};
  if (kind == 0) {
    double den = u1[IX] * c1 + u1[IY] * s1;
    for (int j = 0; j < 6; j++) c[j] = -(u1[IX] * A[IX * 6 + j] + u1[IY] * A[IY * 6 + j]) / den;
  } else {
    c[IZ] = -st / ct;
    c[ITH] = (pos - u[IZ]) / (ct * ct);
  }
  for (int i = 0; i < 6; i++) for (int j = 0; j < 6; j++) F[i * 6 + j] = A[i * 6 + j] + b[i] * c[j];
}

void fcft(const double* F, const double* C, double* out) {
  double T[36];
  for (int i = 0; i < 6; i++) for (int j = 0; j < 6; j++) {
    double acc = 0; for (int k = 0; k < 6; k++) acc += F[i * 6 + k] * C[k * 6 + j]; T[i * 6 + j] = acc; }
  for (int i = 0; i < 6; i++) for (int j = 0; j < 6; j++) {
    double acc = 0; for (int k = 0; k < 6; k++) acc += T[i * 6 + k] * F[j * 6 + k]; out[i * 6 + j] = acc; }
  for (int i = 0; i < 6; i++) for (int j = 0; j < i; j++) {
    double m = 0.5 * (out[i * 6 + j] + out[j * 6 + i]); out[i * 6 + j] = out[j * 6 + i] = m; }
}

int propagate(int kind, double pos, double bz, const State& in, State& out, double* F_out, double* s_out, int dir = 1) {
  double s;
  if (!path_to_surface(kind, pos, bz, in.q, in.u, &s, dir)) return MKFO_PROP_UNREACHABLE;
  helix_step(bz, in.q, in.u, s, out.u);
  double F[36];
  jacobian(kind, pos, bz, in.q, in.u, out.u, s, F);
  fcft(F, in.C, out.C);
  out.q = in.q;
  if (F_out) std::memcpy(F_out, F, sizeof(F));
  if (s_out) *s_out = s;
  return 0;
}

// C5 constants: silicon, pion (DESIGN.md §3 U8).
const double M_PI_GEV = 0.13957039, M_E_GEV = 0.51099895e-3;
const double BB_K = 0.307075e-3;        // GeV cm^2 / mol
const double SI_ZA = 14.0 / 28.0855, SI_RHO = 2.329, SI_I = 173e-9, SI_X0 = 9.37;

double dedx(double p) {                 // -dE/dx [GeV/cm], Bethe-Bloch without density correction
  double m = M_PI_GEV, E = std::sqrt(p * p + m * m), beta = p / E, gamma = E / m;
  double b2g2 = beta * beta * gamma * gamma;
  double tmax = 2.0 * M_E_GEV * b2g2 / (1.0 + 2.0 * gamma * M_E_GEV / m + (M_E_GEV / m) * (M_E_GEV / m));
  return BB_K * SI_ZA * SI_RHO / (beta * beta) *
         (0.5 * std::log(2.0 * M_E_GEV * b2g2 * tmax / (SI_I * SI_I)) - beta * beta);
}
// R12: Gaussian energy-loss straggling, variance of the loss in thickness t (radiation lengths
// along the path): sigma_E^2 = xi Tmax (1 - beta^2/2) with xi = (K/2)(Z/A) rho x / beta^2, x = t X0 (Bohr's variance
// with the relativistic factor; the same Tmax as Bethe-Bloch).
double straggling_var(double p, double t) {
  double m = M_PI_GEV, E = std::sqrt(p * p + m * m), beta2 = p * p / (E * E), gamma = E / m;
  double b2g2 = beta2 * gamma * gamma;
  double tmax = 2.0 * M_E_GEV * b2g2 / (1.0 + 2.0 * gamma * M_E_GEV / m + (M_E_GEV / m) * (M_E_GEV / m));
  double xi = 0.5 * BB_K * SI_ZA * SI_RHO * (t * SI_X0) / beta2;
  return xi * tmax * (1.0 - 0.5 * beta2);
}
double highland(double p, double t) {
  double m = M_PI_GEV, E = std::sqrt(p * p + m * m), beta = p / E;
  return 0.0136 / (beta * p) * std::sqrt(t) * (1.0 + 0.038 * std::log(t));
}

// dir = -1 (R7): the layer is crossed against the particle's motion: the mean energy loss is given back, the
// scattering noise is added all the same; both are evaluated with the momentum the state arrives with.
int material(int kind, double xx0, int flags, double* u, double* C, double* th0_out, double* dE_out, int dir = 1) {
  if (th0_out) *th0_out = 0; if (dE_out) *dE_out = 0;
  if (!(xx0 > 0) || (flags & 3) == 0) return 0;
  double st = std::sin(u[ITH]), ct = std::cos(u[ITH]);
  double pn;                                                     // |p_hat . n_hat|
  if (kind == 0) { double r = std::hypot(u[IX], u[IY]);
    pn = std::fabs(st * (u[IX] * std::cos(u[IPHI]) + u[IY] * std::sin(u[IPHI])) / r); }
  else pn = std::fabs(ct);
  double t = xx0 / pn;
  double aipt = std::fabs(u[IIPT]);
  double p = 1.0 / (aipt * std::fabs(st));
  double m = M_PI_GEV, E = std::sqrt(p * p + m * m), beta = p / E;
  double th0 = highland(p, t);                                   // with p before the energy loss
  if (flags & 2) {
    double dE = dedx(p) * t * SI_X0;
    double E1 = dir > 0 ? E - dE : E + dE;
    if (dE_out) *dE_out = dE;
    if (E1 <= m) return MKFO_STOPPED_ELOSS;
    double p1 = std::sqrt(E1 * E1 - m * m), beta1 = p1 / E1;
    double J = (p / p1) * (p / p1) * (beta / beta1);
    u[IIPT] *= p / p1;
    for (int j = 0; j < 6; j++) { C[IIPT * 6 + j] *= J; }
    for (int j = 0; j < 6; j++) { C[j * 6 + IIPT] *= J; }
    if (flags & 4) {
      // R12: the loss fluctuates with variance sigma_E^2 (evaluated with the momentum the state arrives with); a shift
      // dE of the energy moves ipt by ipt1 (E1 / p1^2) dE at fixed direction
      double k = u[IIPT] * E1 / (p1 * p1);
      C[IIPT * 6 + IIPT] += k * k * straggling_var(p, t);
    }
  }
  if (flags & 1) {
    if (th0_out) *th0_out = th0;
    double t2 = th0 * th0, cot = ct / st, ip = u[IIPT];
    C[IPHI * 6 + IPHI] += t2 / (st * st);
    C[ITH * 6 + ITH] += t2;
    C[IIPT * 6 + IIPT] += ip * ip * cot * cot * t2;
    C[IIPT * 6 + ITH] -= ip * cot * t2;
    C[ITH * 6 + IIPT] -= ip * cot * t2;
  }
  return 0;
}

// 3x3 SPD inverse by Cholesky; false if not positive definite.
bool spd_inverse3(const double* S, double* Sinv) {
  double L[9] = {0};
  for (int i = 0; i < 3; i++) for (int j = 0; j <= i; j++) {
    double acc = S[i * 3 + j];
    for (int k = 0; k < j; k++) acc -= L[i * 3 + k] * L[j * 3 + k];
    if (i == j) { if (!(acc > 0)) return false; L[i * 3 + i] = std::sqrt(acc); }
    else L[i * 3 + j] = acc / L[j * 3 + j];
  }
  double Li[9] = {0};                                            // inverse of lower-triangular L
  for (int i = 0; i < 3; i++) { Li[i * 3 + i] = 1.0 / L[i * 3 + i];
    for (int j = 0; j < i; j++) { double acc = 0; for (int k = j; k < i; k++) acc -= L[i * 3 + k] * Li[k * 3 + j];
      Li[i * 3 + j] = acc / L[i * 3 + i]; } }
  for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) {
    double acc = 0; for (int k = 0; k < 3; k++) acc += Li[k * 3 + i] * Li[k * 3 + j]; Sinv[i * 3 + j] = acc; }
  return true;
}

void unpackV(const double* V6, double* V) {                      // xx,xy,yy,xz,yz,zz -> 3x3
  V[0] = V6[0]; V[1] = V[3] = V6[1]; V[4] = V6[2]; V[2] = V[6] = V6[3]; V[5] = V[7] = V6[4]; V[8] = V6[5];
}

// C6: chi2 = r^T S^-1 r with S = C(0:3,0:3)+V. Optionally the full Joseph-form update.
int chi2_update(double* u, double* C, const double* m, const double* V6, double* chi2, bool do_update) {
  double V[9]; unpackV(V6, V);
  double S[9], Sinv[9], r[3];
  for (int i = 0; i < 3; i++) { r[i] = m[i] - u[i]; for (int j = 0; j < 3; j++) S[i * 3 + j] = C[i * 6 + j] + V[i * 3 + j]; }
  if (!spd_inverse3(S, Sinv)) return MKFO_S_NOT_PD;
  double c2 = 0; for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) c2 += r[i] * Sinv[i * 3 + j] * r[j];
  *chi2 = c2;
  if (!do_update) return 0;
  double K[18];                                                  // 6x3 gain K = C(:,0:3) S^-1
  for (int i = 0; i < 6; i++) for (int j = 0; j < 3; j++) {
    double acc = 0; for (int k = 0; k < 3; k++) acc += C[i * 6 + k] * Sinv[k * 3 + j]; K[i * 3 + j] = acc; }
  for (int i = 0; i < 6; i++) for (int j = 0; j < 3; j++) u[i] += K[i * 3 + j] * r[j];
  double IKH[36];                                                // I - K H, H = [I3 | 0]
  for (int i = 0; i < 6; i++) for (int j = 0; j < 6; j++) IKH[i * 6 + j] = (i == j ? 1.0 : 0.0) - (j < 3 ? K[i * 3 + j] : 0.0);
  double Cn[36]; fcft(IKH, C, Cn);
  for (int i = 0; i < 6; i++) for (int j = 0; j < 6; j++) {      // + K V K^T
    double acc = 0; for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) acc += K[i * 3 + a] * V[a * 3 + b] * K[j * 3 + b];
    Cn[i * 6 + j] += acc; }
  for (int i = 0; i < 6; i++) for (int j = 0; j <= i; j++) { double mm = 0.5 * (Cn[i * 6 + j] + Cn[j * 6 + i]); C[i * 6 + j] = C[j * 6 + i] = mm; }
  return 0;
}

void load_state(int n, int i, const float* par, const float* cov, const signed char* q, State& st) {
  for (int k = 0; k < 6; k++) st.u[k] = (double)par[(size_t)k * n + i];
  for (int a = 0; a < 6; a++) for (int b = 0; b <= a; b++) {
    double v = (double)cov[(size_t)(a * (a + 1) / 2 + b) * n + i]; st.C[a * 6 + b] = st.C[b * 6 + a] = v; }
  st.q = q[i];
}
void store_state(int n, int i, const State& st, double* par, double* cov) {
  for (int k = 0; k < 6; k++) par[(size_t)k * n + i] = st.u[k];
  for (int a = 0; a < 6; a++) for (int b = 0; b <= a; b++) cov[(size_t)(a * (a + 1) / 2 + b) * n + i] = st.C[a * 6 + b];
}
void load_hit(const mkfo_hits* h, int id, double* m, double* V6) {
  m[0] = h->x[id]; m[1] = h->y[id]; m[2] = h->z[id];
  for (int k = 0; k < 6; k++) V6[k] = (double)h->V[(size_t)k * h->n_hits + id];
}

// cos of the incidence angle in the transverse plane (U7) for a state on a barrel surface.
double cos_alpha(const double* u) {
  return (u[IX] * std::cos(u[IPHI]) + u[IY] * std::sin(u[IPHI])) / std::hypot(u[IX], u[IY]);
}

// R13 (SURVEY f4 "non-uniform field hook"; PAPER.md:41 lists the magnetic field among the ingredients of the
// lightweight geometry): the step that ends on layer l runs in the uniform field bz_layer[l].
inline double bz_of(const mkfo_geometry* g, int layer) { return g->bz_layer ? (double)g->bz_layer[layer] : (double)g->bz; }

// One filter step of C7/C9 up to (not including) the update: propagate -> grazing test -> material.
// returns 0, or a status bit. `skip` semantics are decided by the caller.
int step_to_layer(const mkfo_geometry* g, const mkfo_params* p, const mkfo_layer& L, const State& in, State& out) {
  int rc = propagate(L.kind, (double)L.pos, bz_of(g, (int)(&L - g->layers)), in, out, nullptr, nullptr);
  if (rc) return rc;
  if (L.kind == 0) { if (cos_alpha(out.u) < (double)p->graze_cos_min) return MKFO_GRAZING; }
  else { if (std::fabs(std::cos(out.u[ITH])) < DISK_GRAZE_COS) return MKFO_GRAZING; }
  rc = material(L.kind, (double)L.xx0, p->material_flags, out.u, out.C, nullptr, nullptr);
  return rc;
}

bool has_nan(const State& s) {
  for (int k = 0; k < 6; k++) if (!std::isfinite(s.u[k])) return true;
  for (int k = 0; k < 36; k++) if (!std::isfinite(s.C[k])) return true;
  return false;
}

// ---- C8 helpers -------------------------------------------------------------------------------------
int phi_bin(double phi, int nphi) {
  int ip = (int)std::floor((phi + PI) * nphi / (2.0 * PI));
  if (ip >= nphi) ip -= nphi; if (ip < 0) ip = 0; return ip;
}
int eta_bin(double eta, double lo, double hi, int neta) {
  int ie = (int)std::floor((eta - lo) * neta / (hi - lo));
  if (ie < 0) ie = 0; if (ie > neta - 1) ie = neta - 1; return ie;
}

// U11 window.
void window(const mkfo_geometry* g, const mkfo_params* p, int layer, const double* u, const double* C,
            const double* vmax, int* e0, int* e1, int* p0, int* np) {
  const mkfo_layer& L = g->layers[layer];
  int nphi = g->n_phi_bins, neta = g->n_eta_bins;
  double cut = p->chi2_cut, vxy = vmax[0], vzz = vmax[1];
  double x = u[IX], y = u[IY], z = u[IZ], r = std::hypot(x, y);
  double php = std::atan2(y, x);
  double dphi, eta_a, eta_b;
  if (L.kind == 0) {
    double R = L.pos;
    double tx = -y / r, ty = x / r, nx = x / r, ny = y / r;
    double Ctt = tx * tx * C[0] + 2 * tx * ty * C[1] + ty * ty * C[7];
    double Cnn = nx * nx * C[0] + 2 * nx * ny * C[1] + ny * ny * C[7];
    if (Ctt < 0) Ctt = 0; if (Cnn < 0) Cnn = 0;
    double dz = std::sqrt(cut * (C[IZ * 6 + IZ] + vzz));
    double a1 = std::sqrt(cut * (Ctt + vxy)) / R;
    double a2 = std::sqrt(cut * (Cnn + vxy)) / R + 1e-6;
    dphi = a2 < 2.0 ? std::acos(1.0 - a2) : PI;
    if (a1 < 1.0 && dphi <= 0.5 * PI) dphi = std::min(dphi, std::asin(a1));
    eta_a = std::asinh((z - dz) / R); eta_b = std::asinh((z + dz) / R);
  } else {
    double Z = L.pos;
    double rw = std::sqrt(cut * (C[0] + C[7] + vxy));
    dphi = rw < r ? std::asin(rw / r) : PI;
    double rlo = std::max(r - rw, 1e-3), rhi = r + rw;
    double ea = std::asinh(Z / rlo), eb = std::asinh(Z / rhi);
    eta_a = std::min(ea, eb); eta_b = std::max(ea, eb);
  }
  dphi *= 1.0 + 1e-6; dphi += 1e-6;
  *e0 = std::max(0, eta_bin(eta_a, L.eta_lo, L.eta_hi, neta) - 1);
  *e1 = std::min(neta - 1, eta_bin(eta_b, L.eta_lo, L.eta_hi, neta) + 1);
  if (dphi >= PI) { *p0 = 0; *np = nphi; return; }
  double bw = 2.0 * PI / nphi;
  int a = (int)std::floor((php - dphi + PI) / bw) - 1;
  int b = (int)std::floor((php + dphi + PI) / bw) + 1;
  int cnt = b - a + 1;
  if (cnt >= nphi) { *p0 = 0; *np = nphi; return; }
  *p0 = ((a % nphi) + nphi) % nphi; *np = cnt;
}

// ---- C9 bookkeeping -----------------------------------------------------------------------------------
struct Cand {
  State st; double chi2; int nhits, nmiss, consec; unsigned status;
  std::vector<int> hits;                                         // per plan step: id | -1 | -2
  std::vector<int> hits2;                                        // R15: a second hit of the step (overlapping module) | -2
};
struct Child { double score, chi2; int parent; int hit; int kind; /* 0 hit, 1 miss, 2 pass-through */ };
const int HIT_INF = std::numeric_limits<int>::max();

inline double score_of(const mkfo_params* p, int nhits, int nmiss, double chi2) {      // U13
  return (double)p->score_hit * nhits - (double)p->score_miss * nmiss - chi2;
}
// U14 total order: higher score, lower chi2, lower parent rank, lower hit id (miss = +inf).
inline bool child_before(const Child& a, const Child& b) {
  if (a.score != b.score) return a.score > b.score;
  if (a.chi2 != b.chi2) return a.chi2 < b.chi2;
  if (a.parent != b.parent) return a.parent < b.parent;
  return a.hit < b.hit;
}

}  // namespace

// =====================================================================================================
extern "C" {

int mkfo_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void mkfo_helix_step(double bz, int q, const double* u, double s, double* u1) { helix_step(bz, q, u, s, u1); }

int mkfo_propagate(int kind, double pos, double bz, int q, const double* u, const double* C, double* u1,
                   double* F, double* C1, double* s) {
  State in, out; std::memcpy(in.u, u, sizeof(in.u)); in.q = q;
  if (C) std::memcpy(in.C, C, sizeof(in.C)); else std::memset(in.C, 0, sizeof(in.C));
  int rc = propagate(kind, pos, bz, in, out, F, s);
  if (rc) return rc;
  std::memcpy(u1, out.u, sizeof(out.u));
  if (C1) std::memcpy(C1, out.C, sizeof(out.C));
  return 0;
}

int mkfo_material(int kind, double xx0, int flags, double* u, double* C, double* theta0_out, double* dE_out) {
  return material(kind, xx0, flags, u, C, theta0_out, dE_out);
}
int mkfo_propagate_dir(int kind, double pos, double bz, int q, int dir, const double* u, const double* C, double* u1,
                       double* F, double* C1, double* s) {
  State in, out; std::memcpy(in.u, u, sizeof(in.u)); in.q = q;
  if (C) std::memcpy(in.C, C, sizeof(in.C)); else std::memset(in.C, 0, sizeof(in.C));
  int rc = propagate(kind, pos, bz, in, out, F, s, dir);
  if (rc) return rc;
  std::memcpy(u1, out.u, sizeof(out.u));
  if (C1) std::memcpy(C1, out.C, sizeof(out.C));
  return 0;
}
int mkfo_material_dir(int kind, double xx0, int flags, int dir, double* u, double* C, double* theta0_out, double* dE_out) {
  return material(kind, xx0, flags, u, C, theta0_out, dE_out, dir);
}
double mkfo_dedx(double p) { return dedx(p); }
double mkfo_highland(double p, double t) { return highland(p, t); }
double mkfo_straggling_var(double p, double t) { return straggling_var(p, t); }

int mkfo_chi2(const double* u, const double* C, const double* m, const double* V, double* chi2) {
  double uu[6], CC[36]; std::memcpy(uu, u, sizeof(uu)); std::memcpy(CC, C, sizeof(CC));
  return chi2_update(uu, CC, m, V, chi2, false);
}
int mkfo_update(double* u, double* C, const double* m, const double* V, double* chi2) {
  return chi2_update(u, C, m, V, chi2, true);
}
void mkfo_window(const mkfo_geometry* g, const mkfo_params* p, int layer, const double* u, const double* C,
                 const double* vmax, int* e0, int* e1, int* p0, int* np) {
  window(g, p, layer, u, C, vmax, e0, e1, p0, np);
}

// ---- C8 ---------------------------------------------------------------------------------------------
// R9 ("Hits used in tracks reconstructed with high quality are masked to reduce the
// combinatorics of the next iteration"): a masked hit (mask[i] != 0) is left out of the index altogether: it is in
// no bin, it does not count for vmax, and sorted_id holds bin_off[last] < n_hits entries. mask == NULL: C8 as before.
int mkfo_build_hit_index_masked(const mkfo_geometry* g, const mkfo_hits* h, const unsigned char* mask, unsigned* bin_off,
                                int* sorted_id, float* vmax);
int mkfo_build_hit_index(const mkfo_geometry* g, const mkfo_hits* h, unsigned* bin_off, int* sorted_id, float* vmax) {
  return mkfo_build_hit_index_masked(g, h, nullptr, bin_off, sorted_id, vmax);
}
int mkfo_build_hit_index_masked(const mkfo_geometry* g, const mkfo_hits* h, const unsigned char* mask, unsigned* bin_off,
                                int* sorted_id, float* vmax) {
  int nl = g->n_layers, nphi = g->n_phi_bins, neta = g->n_eta_bins, nb = nphi * neta;
  size_t nseg = (size_t)h->n_events * nl;
  std::vector<unsigned> cnt(nseg * nb + 1, 0u);
  std::vector<int> key(h->n_hits, 0);
  for (int ev = 0; ev < h->n_events; ev++) for (int l = 0; l < nl; l++) {
    size_t seg = (size_t)ev * nl + l;
    int b = h->layer_off[ev * (nl + 1) + l], e = h->layer_off[ev * (nl + 1) + l + 1];
    const mkfo_layer& L = g->layers[l];
    float vxy = 0.f, vzz = 0.f;
    for (int i = b; i < e; i++) {
      if (mask && mask[i]) { key[i] = -1; continue; }
      double x = h->x[i], y = h->y[i], z = h->z[i];
      int ip = phi_bin(std::atan2(y, x), nphi);
      int ie = eta_bin(std::asinh(z / std::sqrt(x * x + y * y)), (double)L.eta_lo, (double)L.eta_hi, neta);
      key[i] = ie * nphi + ip;
      cnt[seg * nb + key[i]]++;
      // larger eigenvalue of the xy block of V, in float arithmetic order fixed: see DESIGN.md (U11/C8)
      float vxx = h->V[i], vxyv = h->V[(size_t)h->n_hits + i], vyy = h->V[(size_t)2 * h->n_hits + i];
      float hs = 0.5f * (vxx + vyy), hd = 0.5f * (vxx - vyy);
      float ev1 = hs + sqrtf(hd * hd + vxyv * vxyv);
      if (ev1 > vxy) vxy = ev1;
      float vz = h->V[(size_t)5 * h->n_hits + i];
      if (vz > vzz) vzz = vz;
    }
    vmax[seg * 2] = vxy; vmax[seg * 2 + 1] = vzz;
  }
  unsigned run = 0;
  for (size_t k = 0; k < nseg * nb; k++) { unsigned c = cnt[k]; bin_off[k] = run; run += c; }
  bin_off[nseg * nb] = run;
  std::vector<unsigned> cur(bin_off, bin_off + nseg * nb);
  for (int ev = 0; ev < h->n_events; ev++) for (int l = 0; l < nl; l++) {
    size_t seg = (size_t)ev * nl + l;
    int b = h->layer_off[ev * (nl + 1) + l], e = h->layer_off[ev * (nl + 1) + l + 1];
    for (int i = b; i < e; i++) if (key[i] >= 0) sorted_id[cur[seg * nb + key[i]]++] = i;      // ascending id within a bin
  }
  return 0;
}

// ---- C7 ---------------------------------------------------------------------------------------------
int mkfo_fit(const mkfo_geometry* g, const mkfo_params* p, const mkfo_hits* h, int n, const float* par,
             const float* cov, const signed char* q, const signed char* plan, const int* track_hits,
             int max_plan_len, double* par_out, double* cov_out, double* chi2, int* nfit, unsigned* status) {
#pragma omp parallel for schedule(static)
  for (int i = 0; i < n; i++) {
    State st; load_state(n, i, par, cov, q, st);
    const int* pl = g->plan_layers + g->plan_off[plan[i]];
    int plen = g->plan_off[plan[i] + 1] - g->plan_off[plan[i]];
    double c2tot = 0; int nf = 0; unsigned stat = 0;
    for (int s = 0; s < plen && s < max_plan_len; s++) {
      int hid = track_hits[(size_t)s * n + i];
      if (hid < 0) continue;
      const mkfo_layer& L = g->layers[pl[s]];
      State nx;
      int rc = step_to_layer(g, p, L, st, nx);
      if (rc) { stat |= (unsigned)rc; break; }
      double m[3], V6[6]; load_hit(h, hid, m, V6);
      double c2;
      rc = chi2_update(nx.u, nx.C, m, V6, &c2, true);
      if (rc) { stat |= (unsigned)rc; break; }
      if (has_nan(nx)) { stat |= MKFO_NAN; break; }
      st = nx; c2tot += c2; nf++;
    }
    store_state(n, i, st, par_out, cov_out);
    chi2[i] = c2tot; nfit[i] = nf; status[i] = stat;
  }
  return 0;
}

// ---- R7: backward (outside-in) fit -------------------------------------------------------------------
// PAPER.md:25 "Fitting simply applies the KF procedure to all hits identified during building"; the same
// filter run from the outermost hit inwards gives the parameters at the innermost hit. The seed is a state on the
// outer side of the layer of the track's LAST hit. Per hit, from the last to the first: (not for the first one
// processed) give back the material of the layer just left (C5 with dir = -1), propagate backward to the hit's layer
// (C2/C3 with s <= 0), grazing test (U7), transport (C4), update (C6). A state arriving from outside describes the
// particle on the outer side of the layer (after its scattering there), so the layer's material is given back after
// the update, before moving further in; the result is the state at the innermost hit before that layer's material.
// A track that stops early keeps the state after its last good update (material of that layer not given back).
int mkfo_fit_backward(const mkfo_geometry* g, const mkfo_params* p, const mkfo_hits* h, int n, const float* par,
             const float* cov, const signed char* q, const signed char* plan, const int* track_hits,
             int max_plan_len, double* par_out, double* cov_out, double* chi2, int* nfit, unsigned* status) {
#pragma omp parallel for schedule(static)
  for (int i = 0; i < n; i++) {
    State st; load_state(n, i, par, cov, q, st);
    const int* pl = g->plan_layers + g->plan_off[plan[i]];
    int plen = g->plan_off[plan[i] + 1] - g->plan_off[plan[i]];
    if (plen > max_plan_len) plen = max_plan_len;
    double c2tot = 0; int nf = 0; unsigned stat = 0; int prev = -1;
    for (int s = plen - 1; s >= 0; s--) {
      int hid = track_hits[(size_t)s * n + i];
      if (hid < 0) continue;
      const mkfo_layer& L = g->layers[pl[s]];
      State cur = st;
      if (prev >= 0) {
        const mkfo_layer& Lp = g->layers[prev];
        int rc = material(Lp.kind, (double)Lp.xx0, p->material_flags, cur.u, cur.C, nullptr, nullptr, -1);
        if (rc) { stat |= (unsigned)rc; break; }
      }
      State nx;
      // R13: going back along the arc that the forward step to the layer being left ran on
      int rc = propagate(L.kind, (double)L.pos, bz_of(g, prev >= 0 ? prev : pl[s]), cur, nx, nullptr, nullptr, -1);
      if (rc) { stat |= (unsigned)rc; break; }
      if (L.kind == 0) { if (cos_alpha(nx.u) < (double)p->graze_cos_min) { stat |= MKFO_GRAZING; break; } }
      else { if (std::fabs(std::cos(nx.u[ITH])) < DISK_GRAZE_COS) { stat |= MKFO_GRAZING; break; } }
      double m[3], V6[6]; load_hit(h, hid, m, V6);
      double c2;
      rc = chi2_update(nx.u, nx.C, m, V6, &c2, true);
      if (rc) { stat |= (unsigned)rc; break; }
      if (has_nan(nx)) { stat |= MKFO_NAN; break; }
      st = nx; c2tot += c2; nf++; prev = pl[s];
    }
    // the layer of the innermost fitted hit is given back too: the result is the state BEFORE that layer's material
    // (scattering there is not constrained by any hit further in)
    if (prev >= 0 && stat == 0) {
      const mkfo_layer& Lp = g->layers[prev];
      State cur = st;
      if (material(Lp.kind, (double)Lp.xx0, p->material_flags, cur.u, cur.C, nullptr, nullptr, -1) == 0) st = cur;
    }
    store_state(n, i, st, par_out, cov_out);
    chi2[i] = c2tot; nfit[i] = nf; status[i] = stat;
  }
  return 0;
}

// ---- R14: two-filter smoother -----------------------------------------------------------------
namespace {
// local frame of a surface at point u: rows (in-surface 1, in-surface 2, ipt, phi, theta); barrel: tangential, z;
// disk: x, y. Orthonormal rows; the surface normal is left out (the covariance is null along it, U2).
void local_frame(int kind, const double* u, double* T /* 5x6 */) {
  std::memset(T, 0, 30 * sizeof(double));
  if (kind == 0) { double r = std::hypot(u[IX], u[IY]); T[0 * 6 + IX] = -u[IY] / r; T[0 * 6 + IY] = u[IX] / r; T[1 * 6 + IZ] = 1.0; }
  else { T[0 * 6 + IX] = 1.0; T[1 * 6 + IY] = 1.0; }
  T[2 * 6 + IIPT] = 1.0; T[3 * 6 + IPHI] = 1.0; T[4 * 6 + ITH] = 1.0;
}
// SPD inverse of an n x n matrix by Cholesky (n <= 5); false if not positive definite.
bool spd_inverse(int n, const double* A, double* Ainv) {
  double L[25] = {0}, Li[25] = {0};
  for (int i = 0; i < n; i++) for (int j = 0; j <= i; j++) {
    double acc = A[i * n + j];
    for (int k = 0; k < j; k++) acc -= L[i * n + k] * L[j * n + k];
    if (i == j) { if (!(acc > 0)) return false; L[i * n + i] = std::sqrt(acc); }
    else L[i * n + j] = acc / L[j * n + j];
  }
  for (int i = 0; i < n; i++) { Li[i * n + i] = 1.0 / L[i * n + i];
    for (int j = 0; j < i; j++) { double acc = 0; for (int k = j; k < i; k++) acc -= L[i * n + k] * Li[k * n + j];
      Li[i * n + j] = acc / L[i * n + i]; } }
  for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) {
    double acc = 0; for (int k = 0; k < n; k++) acc += Li[k * n + i] * Li[k * n + j]; Ainv[i * n + j] = acc; }
  return true;
}
bool smooth_combine(int kind, const double* uf, const double* Cf, const double* ub, const double* Cb, double* us, double* Cs) {
  double T[30]; local_frame(kind, uf, T);
  double a[5], Pf[25], Pb[25], M[25], Mi[25], K[25];
  for (int i = 0; i < 5; i++) {
    double acc = 0;
    for (int k = 0; k < 6; k++) { double d = ub[k] - uf[k]; if (k == IPHI) d = std::remainder(d, 2.0 * PI); acc += T[i * 6 + k] * d; }
    a[i] = acc;
  }
  auto project = [&](const double* C, double* P) {
    for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) {
      double acc = 0;
      for (int k = 0; k < 6; k++) for (int l = 0; l < 6; l++) acc += T[i * 6 + k] * C[k * 6 + l] * T[j * 6 + l];
      P[i * 5 + j] = acc; } };
  project(Cf, Pf); project(Cb, Pb);
  for (int i = 0; i < 25; i++) M[i] = Pf[i] + Pb[i];
  if (!spd_inverse(5, M, Mi)) return false;
  for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) { double acc = 0; for (int k = 0; k < 5; k++) acc += Pf[i * 5 + k] * Mi[k * 5 + j]; K[i * 5 + j] = acc; }
  double as[5], Ps[25];
  for (int i = 0; i < 5; i++) { double acc = 0; for (int k = 0; k < 5; k++) acc += K[i * 5 + k] * a[k]; as[i] = acc; }
  // P_s = P_f M P_b (= P_f - P_f M P_f, without the difference of large numbers when one side knows next to nothing)
  for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) { double acc = 0; for (int k = 0; k < 5; k++) acc += K[i * 5 + k] * Pb[k * 5 + j]; Ps[i * 5 + j] = acc; }
  for (int i = 0; i < 5; i++) for (int j = 0; j < i; j++) { double m = 0.5 * (Ps[i * 5 + j] + Ps[j * 5 + i]); Ps[i * 5 + j] = Ps[j * 5 + i] = m; }
  for (int k = 0; k < 6; k++) { double acc = uf[k]; for (int i = 0; i < 5; i++) acc += T[i * 6 + k] * as[i]; us[k] = acc; }
  for (int k = 0; k < 6; k++) for (int l = 0; l < 6; l++) {
    double acc = 0; for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) acc += T[i * 6 + k] * Ps[i * 5 + j] * T[j * 6 + l];
    Cs[k * 6 + l] = acc; }
  return true;
}
}  // namespace

int mkfo_smooth_combine(int kind, const double* u_f, const double* C_f, const double* u_b, const double* C_b, double* u_s, double* C_s) {
  return smooth_combine(kind, u_f, C_f, u_b, C_b, u_s, C_s) ? 0 : MKFO_S_NOT_PD;
}

int mkfo_fit_smooth(const mkfo_geometry* g, const mkfo_params* p, const mkfo_hits* h, int n, const float* par,
             const float* cov, const signed char* q, const signed char* plan, const int* track_hits,
             int max_plan_len, double* par_s, double* cov_s, double* chi2, int* nfit, unsigned* status) {
  std::memset(par_s, 0, sizeof(double) * (size_t)max_plan_len * 6 * n);
  std::memset(cov_s, 0, sizeof(double) * (size_t)max_plan_len * 21 * n);
#pragma omp parallel for schedule(static)
  for (int i = 0; i < n; i++) {
    State st; load_state(n, i, par, cov, q, st);
    const int* pl = g->plan_layers + g->plan_off[plan[i]];
    int plen = std::min(g->plan_off[plan[i] + 1] - g->plan_off[plan[i]], max_plan_len);
    double c2tot = 0; int nf = 0; unsigned stat = 0; bool smoothable = true;
    std::vector<State> pred(plen); std::vector<int> steps;
    // forward filter (C7), keeping the predicted states
    for (int s = 0; s < plen; s++) {
      int hid = track_hits[(size_t)s * n + i];
      if (hid < 0) continue;
      const mkfo_layer& L = g->layers[pl[s]];
      State nx;
      int rc = step_to_layer(g, p, L, st, nx);
      if (rc) { stat |= (unsigned)rc; break; }
      State prd = nx;
      double m[3], V6[6]; load_hit(h, hid, m, V6);
      double c2;
      rc = chi2_update(nx.u, nx.C, m, V6, &c2, true);
      if (rc) { stat |= (unsigned)rc; smoothable = false; break; }
      if (has_nan(nx)) { stat |= MKFO_NAN; smoothable = false; break; }
      pred[s] = prd; steps.push_back(s);
      st = nx; c2tot += c2; nf++;
    }
    chi2[i] = c2tot; nfit[i] = nf; 
    if (smoothable && nf > 0) {
      // backward filter (R7) over the fitted hits, from the forward result with a weak prior
      State cur = st;
      for (int k = 0; k < 36; k++) cur.C[k] *= 1e4;
      std::vector<State> sm(plen); bool ok = true; int prev = -1;
      for (int k = nf - 1; k >= 0 && ok; k--) {
        int s = steps[k];
        const mkfo_layer& L = g->layers[pl[s]];
        State c2s = cur;
        if (prev >= 0) {
          const mkfo_layer& Lp = g->layers[prev];
          int rc = material(Lp.kind, (double)Lp.xx0, p->material_flags, c2s.u, c2s.C, nullptr, nullptr, -1);
          if (rc) { stat |= (unsigned)rc; ok = false; break; }
        }
        State nx;
        int rc = propagate(L.kind, (double)L.pos, bz_of(g, prev >= 0 ? prev : pl[s]), c2s, nx, nullptr, nullptr, -1);
        if (rc) { stat |= (unsigned)rc; ok = false; break; }
        if (L.kind == 0) { if (cos_alpha(nx.u) < (double)p->graze_cos_min) { stat |= MKFO_GRAZING; ok = false; break; } }
        else { if (std::fabs(std::cos(nx.u[ITH])) < DISK_GRAZE_COS) { stat |= MKFO_GRAZING; ok = false; break; } }
        double m[3], V6[6], c2; load_hit(h, track_hits[(size_t)s * n + i], m, V6);
        rc = chi2_update(nx.u, nx.C, m, V6, &c2, true);
        if (rc) { stat |= (unsigned)rc; ok = false; break; }
        if (has_nan(nx)) { stat |= MKFO_NAN; ok = false; break; }
        State out; out.q = nx.q;
        if (!smooth_combine(L.kind, pred[s].u, pred[s].C, nx.u, nx.C, out.u, out.C)) { stat |= MKFO_S_NOT_PD; ok = false; break; }
        sm[s] = out;
        cur = nx; prev = pl[s];
      }
      if (ok) for (int k = 0; k < nf; k++) {
        int s = steps[k];
        for (int a = 0; a < 6; a++) par_s[((size_t)s * 6 + a) * n + i] = sm[s].u[a];
        for (int a = 0; a < 6; a++) for (int b = 0; b <= a; b++) cov_s[((size_t)s * 21 + a * (a + 1) / 2 + b) * n + i] = sm[s].C[a * 6 + b];
      }
    }
    status[i] = stat;
  }
  return 0;
}

// ---- C9 ---------------------------------------------------------------------------------------------
}  // extern "C"
namespace {
// R15 ("the recovery of hits in overlapping detector modules, so that more than one hit per layer
// can be assigned to tracks"): with `module` given (module id per hit; overlapping modules of a layer sit on the same
// surface of the lightweight geometry), a child that took hit h1 on a layer may take ONE more hit of that layer: h2 is
// looked for among its parent's N_c best hits of the layer (by chi2 against the propagated state, the list the
// selection works on) that rank after h1 in that list, with module[h2] != module[h1]; its chi2 against the state already updated with h1 (C6:
// no propagation, no material) must be below the cut; the smallest such chi2 wins (first in list order on a tie). The
// state is updated again, chi2 += chi2_2, nhits += 1 (so the score gains score_hit - chi2_2); an update that does not
// stay finite is not taken. The ranking of the layer itself (C9.6) is done on the first hits alone.
int build_tracks_impl(const mkfo_geometry* g, const mkfo_params* p, const mkfo_hits* h, const unsigned* bin_off,
             const int* sorted_id, const float* vmax, int brute_force, int n, const float* par,
             const float* cov, const signed char* q, const int* seed_event, const int* seed_hits,
             const signed char* plan, int max_plan_len, double* par_out, double* cov_out, double* chi2,
             double* score, int* nhits, int* nmiss, int* hit_ids, unsigned* status, double* margin,
             long long* n_chi2_evals, const int* module, int* hit_ids2) {
  int nl = g->n_layers, nphi = g->n_phi_bins, neta = g->n_eta_bins, nb = nphi * neta;
  long long evals_total = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : evals_total)
  for (int i = 0; i < n; i++) {
    const int* pl = g->plan_layers + g->plan_off[plan[i]];
    int plen = std::min(g->plan_off[plan[i] + 1] - g->plan_off[plan[i]], max_plan_len);
    int ev = seed_event[i];
    const int* loff = h->layer_off + (size_t)ev * (nl + 1);
    double mrg = std::numeric_limits<double>::infinity();
    auto note = [&](double m) { m = std::fabs(m); if (m < mrg) mrg = m; };

    // seed candidate: fit the seed state through its own three hits (reading U18b)
    Cand seed; load_state(n, i, par, cov, q, seed.st);
    seed.chi2 = 0; seed.nhits = 0; seed.nmiss = 0; seed.consec = 0; seed.status = 0;
    seed.hits.assign(max_plan_len, -2); seed.hits2.assign(max_plan_len, -2);
    int last_step = -1; bool seed_ok = true;
    for (int k = 0; k < 3 && seed_ok; k++) {
      int hid = seed_hits[(size_t)k * n + i];
      int lay = -1;
      for (int l = 0; l < nl; l++) if (hid >= loff[l] && hid < loff[l + 1]) { lay = l; break; }
      int step = -1;
      for (int s = last_step + 1; s < plen; s++) if (pl[s] == lay) { step = s; break; }
      if (step < 0) { seed.status |= MKFO_TRUNCATED; seed_ok = false; break; }
      State nx;
      int rc = step_to_layer(g, p, g->layers[lay], seed.st, nx);
      if (rc) { seed.status |= (unsigned)rc; seed_ok = false; break; }
      double m[3], V6[6], c2; load_hit(h, hid, m, V6);
      rc = chi2_update(nx.u, nx.C, m, V6, &c2, true);
      if (rc) { seed.status |= (unsigned)rc; seed_ok = false; break; }
      seed.st = nx; seed.chi2 += c2; seed.nhits++; seed.hits[step] = hid; last_step = step;
    }

    std::vector<Cand> live; Cand best_short; bool have_short = false;
    auto rank_before = [&](const Cand& a, const Cand& b) {       // U14 on whole candidates
      double sa = score_of(p, a.nhits, a.nmiss, a.chi2), sb = score_of(p, b.nhits, b.nmiss, b.chi2);
      if (sa != sb) return sa > sb; return a.chi2 < b.chi2; };
    auto offer_short = [&](const Cand& c) {
      if (c.nhits < p->min_hits_keep) return;
      if (!have_short || rank_before(c, best_short)) { best_short = c; have_short = true; } };
    if (seed_ok) live.push_back(seed);

    for (int s = last_step + 1; s < plen && seed_ok && !live.empty(); s++) {
      int lay = pl[s];
      const mkfo_layer& L = g->layers[lay];
      int hb = loff[lay], he = loff[lay + 1];
      size_t seg = (size_t)ev * nl + lay;
      std::vector<Child> pool; std::vector<State> prop(live.size()); std::vector<std::vector<double>> upd_chi2;
      for (int c = 0; c < (int)live.size(); c++) {
        Cand& cd = live[c];
        State nx;
        int rc = propagate(L.kind, (double)L.pos, bz_of(g, lay), cd.st, nx, nullptr, nullptr);
        bool skip = rc != 0;
        if (!skip) {                                             // acceptance (C9.1)
          double v = L.kind == 0 ? nx.u[IZ] : std::hypot(nx.u[IX], nx.u[IY]);
          double ext = (double)L.hi - (double)L.lo;
          note((v - L.lo) / ext); note((L.hi - v) / ext);
          if (v < L.lo || v > L.hi) skip = true;
        }
        if (skip) {                                              // silent skip: unchanged, competes as is
          pool.push_back({score_of(p, cd.nhits, cd.nmiss, cd.chi2), cd.chi2, c, HIT_INF, 2});
          continue;
        }
        bool graze;
        if (L.kind == 0) { double ca = cos_alpha(nx.u); note(ca - p->graze_cos_min); graze = ca < (double)p->graze_cos_min; }
        else { double ca = std::fabs(std::cos(nx.u[ITH])); note(ca - DISK_GRAZE_COS); graze = ca < DISK_GRAZE_COS; }
        if (graze) { cd.status |= MKFO_GRAZING; offer_short(cd); continue; }
        rc = material(L.kind, (double)L.xx0, p->material_flags, nx.u, nx.C, nullptr, nullptr);
        if (rc) { cd.status |= (unsigned)rc; offer_short(cd); continue; }
        prop[c] = nx;
        // candidate hits (C9.3)
        std::vector<int> cands;
        if (brute_force) { for (int id = hb; id < he; id++) cands.push_back(id); }
        else {
          double vm[2] = {(double)vmax[seg * 2], (double)vmax[seg * 2 + 1]};
          int e0, e1, p0, np; window(g, p, lay, nx.u, nx.C, vm, &e0, &e1, &p0, &np);
          for (int ie = e0; ie <= e1; ie++) for (int k = 0; k < np; k++) {
            int ip = (p0 + k) % nphi; size_t bin = seg * nb + (size_t)ie * nphi + ip;
            for (unsigned t = bin_off[bin]; t < bin_off[bin + 1]; t++) cands.push_back(sorted_id[t]);
          }
        }
        for (int id : cands) {
          double m[3], V6[6], c2; load_hit(h, id, m, V6);
          evals_total++;
          if (chi2_update(nx.u, nx.C, m, V6, &c2, false)) continue;
          note((c2 - p->chi2_cut) / p->chi2_cut);
          if (c2 < (double)p->chi2_cut)
            pool.push_back({score_of(p, cd.nhits + 1, cd.nmiss, cd.chi2 + c2), cd.chi2 + c2, c, id, 0});
        }
        pool.push_back({score_of(p, cd.nhits, cd.nmiss + 1, cd.chi2), cd.chi2, c, HIT_INF, 1});   // miss child
      }
      // stopped miss children leave the pool before ranking (C9.5)
      std::vector<Child> ranked;
      for (const Child& ch : pool) {
        if (ch.kind == 1 && live[ch.parent].consec + 1 >= p->max_consec_miss) {
          Cand c = live[ch.parent]; c.st = prop[ch.parent]; c.nmiss++; c.consec++; c.hits[s] = -1;
          offer_short(c);
        } else ranked.push_back(ch);
      }
      std::sort(ranked.begin(), ranked.end(), child_before);
      const std::vector<Child>& ranked_all = ranked;              // within one parent: ascending chi2, then hit id
      int nc = p->max_cand;
      if ((int)ranked.size() > nc) note((ranked[nc - 1].score - ranked[nc].score) / p->score_hit);
      std::vector<Cand> next;
      for (int k = 0; k < (int)ranked.size() && k < nc; k++) {
        const Child& ch = ranked[k];
        Cand c = live[ch.parent];
        if (ch.kind == 2) { c.hits[s] = -2; }
        else if (ch.kind == 1) { c.st = prop[ch.parent]; c.nmiss++; c.consec++; c.hits[s] = -1; }
        else {
          c.st = prop[ch.parent];
          double m[3], V6[6], c2; load_hit(h, ch.hit, m, V6);
          chi2_update(c.st.u, c.st.C, m, V6, &c2, true);
          c.chi2 += c2; c.nhits++; c.consec = 0; c.hits[s] = ch.hit;
          if (has_nan(c.st)) { c.status |= MKFO_NAN; offer_short(live[ch.parent]); continue; }
          if (module) {                                          // R15: one more hit from an overlapping module
            std::vector<Child> plist;                            // the parent's hits of this layer, best first
            for (const Child& o2 : ranked_all) if (o2.kind == 0 && o2.parent == ch.parent) plist.push_back(o2);
            int best = -1; double best_c2 = 0; bool after = false;
            for (int k2 = 0; k2 < (int)plist.size() && k2 < nc; k2++) {
              int h2 = plist[k2].hit;
              if (h2 == ch.hit) { after = true; continue; }
              // only hits that rank AFTER the first one in the parent's list: the pair (h1, h2) is then made once, by the
              // child of its better hit (the other order would give the same state and a twin candidate)
              if (!after || module[h2] == module[ch.hit]) continue;
              double m2[3], V62[6], c2b; load_hit(h, h2, m2, V62);
              if (chi2_update(c.st.u, c.st.C, m2, V62, &c2b, false)) continue;
              if (!(c2b < (double)p->chi2_cut)) continue;
              note((c2b - p->chi2_cut) / p->chi2_cut);
              if (best < 0 || c2b < best_c2) { best = h2; best_c2 = c2b; }
            }
            if (best >= 0) {
              State s2 = c.st;
              double m2[3], V62[6], c2b; load_hit(h, best, m2, V62);
              chi2_update(s2.u, s2.C, m2, V62, &c2b, true);
              if (!has_nan(s2)) { c.st = s2; c.chi2 += c2b; c.nhits++; c.hits2[s] = best; }
            }
          }
        }
        next.push_back(c);
      }
      live.swap(next);
    }
    // final choice: best of live U {best_short}
    const Cand* win = nullptr;
    std::vector<const Cand*> fin;
    for (const Cand& c : live) if (c.nhits >= p->min_hits_keep) fin.push_back(&c);
    if (have_short) fin.push_back(&best_short);
    std::stable_sort(fin.begin(), fin.end(), [&](const Cand* a, const Cand* b) { return rank_before(*a, *b); });
    if (!fin.empty()) { win = fin[0];
      if (fin.size() > 1) note((score_of(p, fin[0]->nhits, fin[0]->nmiss, fin[0]->chi2) -
                                score_of(p, fin[1]->nhits, fin[1]->nmiss, fin[1]->chi2)) / p->score_hit); }
    Cand out = win ? *win : seed;
    if (!win) out.status |= MKFO_TRUNCATED;
    store_state(n, i, out.st, par_out, cov_out);
    chi2[i] = out.chi2; score[i] = score_of(p, out.nhits, out.nmiss, out.chi2);
    nhits[i] = out.nhits; nmiss[i] = out.nmiss; status[i] = out.status; margin[i] = mrg;
    for (int s = 0; s < max_plan_len; s++) hit_ids[(size_t)s * n + i] = out.hits[s];
    if (hit_ids2) for (int s = 0; s < max_plan_len; s++) hit_ids2[(size_t)s * n + i] = out.hits2[s];
  }
  if (n_chi2_evals) *n_chi2_evals = evals_total;
  return 0;
}
}  // namespace
extern "C" {
int mkfo_build_tracks(const mkfo_geometry* g, const mkfo_params* p, const mkfo_hits* h, const unsigned* bin_off,
             const int* sorted_id, const float* vmax, int brute_force, int n, const float* par,
             const float* cov, const signed char* q, const int* seed_event, const int* seed_hits,
             const signed char* plan, int max_plan_len, double* par_out, double* cov_out, double* chi2,
             double* score, int* nhits, int* nmiss, int* hit_ids, unsigned* status, double* margin,
             long long* n_chi2_evals) {
  return build_tracks_impl(g, p, h, bin_off, sorted_id, vmax, brute_force, n, par, cov, q, seed_event, seed_hits, plan, max_plan_len,
                           par_out, cov_out, chi2, score, nhits, nmiss, hit_ids, status, margin, n_chi2_evals, nullptr, nullptr);
}
int mkfo_build_tracks_overlap(const mkfo_geometry* g, const mkfo_params* p, const mkfo_hits* h, const unsigned* bin_off,
             const int* sorted_id, const float* vmax, int brute_force, int n, const float* par,
             const float* cov, const signed char* q, const int* seed_event, const int* seed_hits,
             const signed char* plan, int max_plan_len, double* par_out, double* cov_out, double* chi2,
             double* score, int* nhits, int* nmiss, int* hit_ids, unsigned* status, double* margin,
             long long* n_chi2_evals, const int* module, int* hit_ids2) {
  return build_tracks_impl(g, p, h, bin_off, sorted_id, vmax, brute_force, n, par, cov, q, seed_event, seed_hits, plan, max_plan_len,
                           par_out, cov_out, chi2, score, nhits, nmiss, hit_ids, status, margin, n_chi2_evals, module, hit_ids2);
}

// ---- C10 --------------------------------------------------------------------------------------------
int mkfo_remove_duplicates(const mkfo_params* p, int n_events, const int* track_off, const int* hit_ids,
             int max_plan_len, const int* nhits, const float* score, unsigned char* keep, int* n_kept) {
  int n = track_off[n_events];
#pragma omp parallel for schedule(dynamic, 1)
  for (int ev = 0; ev < n_events; ev++) {
    int b = track_off[ev], e = track_off[ev + 1], kept = 0;
    // hit-id range of this event's tracks, for a membership table (|ids_i ∩ ids_j| by direct lookup)
    int lo = std::numeric_limits<int>::max(), hi = -1;
    for (int i = b; i < e; i++) for (int a = 0; a < max_plan_len; a++) { int ha = hit_ids[(size_t)a * n + i];
      if (ha >= 0) { lo = std::min(lo, ha); hi = std::max(hi, ha); } }
    std::vector<unsigned char> mark(hi >= lo ? (size_t)(hi - lo + 1) : 0, 0);
    for (int i = b; i < e; i++) {
      for (int a = 0; a < max_plan_len; a++) { int ha = hit_ids[(size_t)a * n + i]; if (ha >= 0) mark[ha - lo] = 1; }
      bool removed = false;
      for (int j = b; j < e && !removed; j++) {
        if (j == i) continue;
        int shared = 0;
        for (int c = 0; c < max_plan_len; c++) { int hc = hit_ids[(size_t)c * n + j]; if (hc >= 0 && mark[hc - lo]) shared++; }
        int mn = std::min(nhits[i], nhits[j]);
        if (mn <= 0) continue;
        // shared/mn > dup_frac, evaluated in double on the float parameter
        if ((double)shared > (double)p->dup_frac * (double)mn &&
            (score[j] > score[i] || (score[j] == score[i] && j < i))) removed = true;
      }
      for (int a = 0; a < max_plan_len; a++) { int ha = hit_ids[(size_t)a * n + i]; if (ha >= 0) mark[ha - lo] = 0; }
      keep[i] = removed ? 0 : 1; kept += removed ? 0 : 1;
    }
    n_kept[ev] = kept;
  }
  return 0;
}

// ---- R8: strip clustering (section 4) --------------------------------------------
// "first, seed strips with ADC values greater than 3 times the expected noise are identified; second, clusters are
// formed adding to the seed all strips with ADC values above twice the expected noise that are either consecutive or
// have a small gap (the size of the allowed gap depends on the presence of bad strips in the module); finally, the
// cluster is required to have a quadrature sum of the strip ADCs larger than 5 times the quadrature sum of the
// expected noise, and to have a minimum total charge."
// Reading R8: a bad strip never passes a threshold; consecutive passing strips i < j of one module belong to the same
// cluster iff at most max_holes good strips and at most max_bad bad strips lie strictly between them; a cluster is
// kept iff it holds a seed strip, sum(adc^2) > clus_thr^2 * sum(noise^2) (over its passing strips, fp64, strip order)
// and sum(adc) >= min_charge. Strip thresholds are compared in fp32: (float)adc > thr * noise.
// Output, ordered by (module, first strip): module, first strip and last strip (index inside the module), charge,
// barycentre = sum(adc * (strip + 0.5)) / sum(adc) (fp64, strip order, stored as float). Returns the number kept.
int mkfo_cluster_strips(int n_modules, const int* module_off, const unsigned short* adc, const float* noise,
                        const unsigned char* bad, float seed_thr, float chan_thr, float clus_thr, int min_charge,
                        int max_holes, int max_bad, int* out_module, int* out_first, int* out_last,
                        unsigned* out_charge, float* out_bary) {
  int nout = 0;
  for (int m = 0; m < n_modules; m++) {
    int b = module_off[m], e = module_off[m + 1];
    int i = b;
    while (i < e) {
      bool pass_i = !bad[i] && (float)adc[i] > chan_thr * noise[i];
      if (!pass_i) { i++; continue; }
      // grow the cluster from strip i
      int first = i, last = i;
      bool seed = false; unsigned long long q2 = 0; double n2 = 0, wsum = 0; unsigned charge = 0;
      int j = i, holes = 0, nbad = 0;
      while (j < e) {
        bool pj = !bad[j] && (float)adc[j] > chan_thr * noise[j];
        if (pj) {
          last = j; holes = 0; nbad = 0;
          if ((float)adc[j] > seed_thr * noise[j]) seed = true;
          q2 += (unsigned long long)adc[j] * adc[j]; n2 += (double)noise[j] * (double)noise[j];
          charge += adc[j]; wsum += (double)adc[j] * ((double)(j - b) + 0.5);
        } else {
          if (bad[j]) nbad++; else holes++;
          if (holes > max_holes || nbad > max_bad) break;
        }
        j++;
      }
      if (seed && (double)q2 > (double)clus_thr * (double)clus_thr * n2 && (long long)charge >= (long long)min_charge) {
        out_module[nout] = m; out_first[nout] = first - b; out_last[nout] = last - b; out_charge[nout] = charge;
        out_bary[nout] = (float)(wsum / (double)charge);
        nout++;
      }
      i = last + 1;
    }
  }
  return nout;
}

// ---- R9: which hits the next iteration no longer sees ------------------------------
// The paper does not say what "high quality" is. Reading R9: a track is of high quality iff it survived duplicate
// removal (keep[i] != 0; keep == NULL: every track), has nhits[i] >= min_hits, and chi2[i] <= max_chi2_ndf * ndf with
// ndf = 2 nhits - 5 (two measured coordinates per hit, five parameters), compared in fp32 as the kernel does.
// mask[h] is set to 1 for every hit (id >= 0) of such a track; other entries are left as they are, so that masks
// accumulate over iterations.
int mkfo_mask_hits(int n, int n_hits, const int* hit_ids, int max_plan_len, const int* nhits, const float* chi2,
                   const unsigned char* keep, int min_hits, float max_chi2_ndf, unsigned char* mask) {
  for (int i = 0; i < n; i++) {
    if (keep && !keep[i]) continue;
    if (nhits[i] < min_hits) continue;
    const float ndf = (float)(2 * nhits[i] - 5);
    if (!(chi2[i] <= max_chi2_ndf * ndf)) continue;
    for (int s = 0; s < max_plan_len; s++) {
      const int hid = hit_ids[(size_t)s * n + i];
      if (hid >= 0 && hid < n_hits) mask[hid] = 1;
    }
  }
  return 0;
}

}  // extern "C"
