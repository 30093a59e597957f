// gp_oracle.cpp — TEST INFRASTRUCTURE, not the product.  See gp_oracle.h for the pin list.
//
// Plain scalar double-precision reference for the null-geodesic hot path of arXiv 2310.15183.
// Every function cites the passage of /root/reference/PAPER.md ("P:Lnnn") or the DESIGN.md
// reading ("Rn") it follows.  No blocking, fusion or reordering beyond what those state.
// Build: g++ -O2 -ffp-contract=off -fcx-limited-range -fopenmp -shared -fPIC (oracle/build.py).
//
// Shares nothing with the CUDA library.  Parity unpinned: Manko-Novikov chaotic-set exit
// angles and MAXSTEPS ray states (statistical comparison only).

#include "gp_oracle.h"

#include <cmath>
#include <complex>
#include <cstring>
#include <limits>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

typedef std::complex<double> cplx;
const double kPi = 3.14159265358979323846;
const double kHalfPi = 0.5 * kPi;

// ------------------------------------------------------------------------------------------
// Covariant metrics, generic in the scalar type so that the same literal formulas serve plain
// evaluation (double) and complex-step differentiation (std::complex<double>).
// out: g_tt, g_tphi, g_phiphi, g_rr, g_thth
// ------------------------------------------------------------------------------------------

// P:L136 (eq 8): ds^2 = -(1-2M/r)dt^2 + (1-2M/r)^-1 dr^2 + r^2 dtheta^2 + r^2 sin^2theta dphi^2
template <class T>
void schwarzschild_cov(double M, T r, T th, T g[5]) {
  T F = 1.0 - 2.0 * M / r;
  T s = std::sin(th);
  g[0] = -F;
  g[1] = T(0.0);
  g[2] = r * r * s * s;
  g[3] = 1.0 / F;
  g[4] = r * r;
}

// P:L147-159 (eq 9-14) with R2 (g_tt has rho^2) and R3 (g_tphi = -2 M a r sin^2theta / rho^2).
template <class T>
void kerr_cov(double M, double a, T r, T th, T g[5]) {
  T s = std::sin(th), c = std::cos(th);
  T rho2 = r * r + a * a * c * c;       // eq 13
  T Delta = r * r - 2.0 * M * r + a * a;  // eq 12
  g[0] = -(1.0 - 2.0 * M * r / rho2);     // eq 9
  g[1] = -2.0 * M * a * r * s * s / rho2; // eq 10 (sign: R3)
  g[2] = s * s / rho2 * ((r * r + a * a) * (r * r + a * a) - a * a * Delta * s * s);  // eq 11
  g[3] = rho2 / Delta;                    // eq 9
  g[4] = rho2;                            // eq 9
}

struct MNConst {
  double M, a, q, alpha, k, beta;
};

// P:L192-196 (eq 23-25) with R7: a = S/M.
MNConst mn_constants(double M, double a, double q) {
  MNConst c;
  c.M = M;
  c.a = a;
  c.q = q;
  c.alpha = (-M + std::sqrt(M * M - a * a)) / a;                 // eq 23
  c.k = M * (1.0 - c.alpha * c.alpha) / (1.0 + c.alpha * c.alpha);  // eq 24
  c.beta = q * M * M * M / (c.k * c.k * c.k);                    // eq 25
  return c;
}

template <class T>
struct MNPot {
  T f, omega, e2gamma, A, B, C, afr, bfr, psi, gammap, rho2, Delta;
};

// P:L186-230 (eq 21-39) with R5 (B), R6 (gamma').
template <class T>
MNPot<T> mn_potentials(const MNConst &c, T r, T th) {
  MNPot<T> o;
  const double al = c.alpha, k = c.k, be = c.beta;
  T x = (r - c.M) / k;    // eq 38
  T y = std::cos(th);     // eq 39
  T R = std::sqrt(x * x + y * y - 1.0);  // eq 36
  T u = x * y / R;                       // eq 37
  T P[4];
  P[0] = T(1.0);
  P[1] = u;
  P[2] = (3.0 * u * u - 1.0) / 2.0;
  P[3] = (5.0 * u * u * u - 3.0 * u) / 2.0;
  T Rp[4];  // R^(l+1)
  Rp[0] = R;
  Rp[1] = R * R;
  Rp[2] = R * R * R;
  o.psi = be * P[2] / Rp[2];  // eq 32
  // eq 34: a = -alpha exp(-2 beta (-1 + sum_l (x-y) P_l / R^(l+1)))
  T Sa = T(0.0), Sb = T(0.0), Sg = T(0.0);
  for (int l = 0; l <= 2; ++l) {
    double sgn_b = ((3 - l) % 2 == 0) ? 1.0 : -1.0;  // (-1)^(3-l)
    double sgn_g = ((2 - l) % 2 == 0) ? 1.0 : -1.0;  // (-1)^(2-l)
    Sa += (x - y) * P[l] / Rp[l];
    Sb += sgn_b * (x + y) * P[l] / Rp[l];
    Sg += (x - y + sgn_g * (x + y)) * P[l] / Rp[l];
  }
  o.afr = -al * std::exp(-2.0 * be * (-1.0 + Sa));  // eq 34
  o.bfr = al * std::exp(2.0 * be * (1.0 + Sb));     // eq 35
  // eq 33 (R6): gamma' = 1/2 ln[(x^2-1)/(x^2-y^2)] + 3 beta^2/(2 R^6) (P3^2 - P2^2) + beta(-2 + Sg)
  T R6 = Rp[2] * Rp[2];
  o.gammap = 0.5 * std::log((x * x - 1.0) / (x * x - y * y)) +
             3.0 * be * be / (2.0 * R6) * (P[3] * P[3] - P[2] * P[2]) + be * (-2.0 + Sg);
  T ab = o.afr * o.bfr;
  T bma = o.bfr - o.afr;
  // eq 29
  o.A = (x * x - 1.0) * (1.0 + ab) * (1.0 + ab) - (1.0 - y * y) * bma * bma;
  // eq 30 (R5)
  T B1 = (x + 1.0) + (x - 1.0) * ab;
  T B2 = (1.0 + y) * o.afr + (1.0 - y) * o.bfr;
  o.B = B1 * B1 + B2 * B2;
  // eq 31
  o.C = (x * x - 1.0) * (1.0 + ab) * (bma - y * (o.afr + o.bfr)) +
        (1.0 - y * y) * bma * ((1.0 + ab) + x * (1.0 - ab));
  o.f = std::exp(2.0 * o.psi) * o.A / o.B;                                             // eq 26
  o.omega = 2.0 * k * std::exp(-2.0 * o.psi) * o.C / o.A - 4.0 * k * al / (1.0 - al * al);  // eq 27
  o.e2gamma = std::exp(2.0 * o.gammap) * o.A / ((x * x - 1.0) * (1.0 - al * al) * (1.0 - al * al));  // eq 28
  T c_ = std::cos(th);
  o.rho2 = (r - c.M) * (r - c.M) - k * k * c_ * c_;  // eq 21
  o.Delta = (r - c.M) * (r - c.M) - k * k;           // eq 22
  return o;
}

// P:L181 (eq 20) with R4:
// ds^2 = -f (dt - omega dphi)^2 + e^{2gamma} rho^2/(f Delta) dr^2 + e^{2gamma} rho^2/f dtheta^2
//        + Delta sin^2theta / f dphi^2
template <class T>
void mn_cov(const MNConst &c, T r, T th, T g[5]) {
  MNPot<T> o = mn_potentials<T>(c, r, th);
  T s = std::sin(th);
  g[0] = -o.f;
  g[1] = o.f * o.omega;
  g[2] = -o.f * o.omega * o.omega + o.Delta * s * s / o.f;
  g[3] = o.e2gamma * o.rho2 / (o.f * o.Delta);
  g[4] = o.e2gamma * o.rho2 / o.f;
}

template <class T>
int metric_cov(const orc_metric *m, T r, T th, T g[5]) {
  switch (m->id) {
    case 0:
      schwarzschild_cov<T>(m->M, r, th, g);
      return 0;
    case 1:
      kerr_cov<T>(m->M, m->a, r, th, g);
      return 0;
    case 2: {
      MNConst c = mn_constants(m->M, m->a, m->q);
      mn_cov<T>(c, r, th, g);
      return 0;
    }
  }
  return -1;
}

// Inverse of a metric whose only off-diagonal entry is g_tphi.
// out: g^tt, g^tphi, g^phiphi, g^rr, g^thth
template <class T>
void invert_block(const T g[5], T gi[5]) {
  T det = g[0] * g[2] - g[1] * g[1];
  gi[0] = g[2] / det;
  gi[1] = -g[1] / det;
  gi[2] = g[0] / det;
  gi[3] = 1.0 / g[3];
  gi[4] = 1.0 / g[4];
}

// Complex-step derivative: Im f(x + i eps)/eps, exact to rounding for analytic f.
int metric_inv_complex_step(const orc_metric *m, double r, double th, double out[15]) {
  const double eps = 1e-30;
  cplx g[5], gi[5];
  if (metric_cov<cplx>(m, cplx(r, eps), cplx(th, 0.0), g)) return -1;
  invert_block<cplx>(g, gi);
  for (int i = 0; i < 5; ++i) {
    out[i] = gi[i].real();
    out[5 + i] = gi[i].imag() / eps;
  }
  metric_cov<cplx>(m, cplx(r, 0.0), cplx(th, eps), g);
  invert_block<cplx>(g, gi);
  for (int i = 0; i < 5; ++i) out[10 + i] = gi[i].imag() / eps;
  return 0;
}

// Schwarzschild inverse metric, each component and derivative written out (from eq 8).
void schwarzschild_inv(double M, double r, double th, double o[15]) {
  double s = std::sin(th), c = std::cos(th);
  double F = 1.0 - 2.0 * M / r;
  double Fr = 2.0 * M / (r * r);
  for (int i = 0; i < 15; ++i) o[i] = 0.0;
  o[0] = -1.0 / F;
  o[2] = 1.0 / (r * r * s * s);
  o[3] = F;
  o[4] = 1.0 / (r * r);
  o[5 + 0] = Fr / (F * F);
  o[5 + 2] = -2.0 / (r * r * r * s * s);
  o[5 + 3] = Fr;
  o[5 + 4] = -2.0 / (r * r * r);
  o[10 + 2] = -2.0 * c / (r * r * s * s * s);
}

// Kerr inverse metric in Boyer-Lindquist coordinates, each component and each of its r, theta
// derivatives written out separately by the quotient rule (inverse of eq 9-13 with R2, R3):
//   g^tt = -Acal/(Sigma Delta), g^tphi = -2 M a r/(Sigma Delta),
//   g^phiphi = (Delta - a^2 s^2)/(Sigma Delta s^2), g^rr = Delta/Sigma, g^thth = 1/Sigma,
//   Acal = (r^2+a^2)^2 - a^2 Delta s^2.
void kerr_inv(double M, double a, double r, double th, double o[15]) {
  double s = std::sin(th), c = std::cos(th);
  double a2 = a * a;
  double Sig = r * r + a2 * c * c;
  double Sig_r = 2.0 * r;
  double Sig_t = -2.0 * a2 * s * c;
  double Del = r * r - 2.0 * M * r + a2;
  double Del_r = 2.0 * r - 2.0 * M;
  double Ac = (r * r + a2) * (r * r + a2) - a2 * Del * s * s;
  double Ac_r = 4.0 * r * (r * r + a2) - a2 * s * s * Del_r;
  double Ac_t = -2.0 * a2 * Del * s * c;
  double D = Sig * Del;
  double D_r = Sig_r * Del + Sig * Del_r;
  double D_t = Sig_t * Del;
  // g^tt
  o[0] = -Ac / D;
  o[5] = -(Ac_r * D - Ac * D_r) / (D * D);
  o[10] = -(Ac_t * D - Ac * D_t) / (D * D);
  // g^tphi
  o[1] = -2.0 * M * a * r / D;
  o[6] = -2.0 * M * a * (D - r * D_r) / (D * D);
  o[11] = 2.0 * M * a * r * D_t / (D * D);
  // g^phiphi
  double n = Del - a2 * s * s;
  double n_r = Del_r;
  double n_t = -2.0 * a2 * s * c;
  double d = D * s * s;
  double d_r = D_r * s * s;
  double d_t = D_t * s * s + 2.0 * D * s * c;
  o[2] = n / d;
  o[7] = (n_r * d - n * d_r) / (d * d);
  o[12] = (n_t * d - n * d_t) / (d * d);
  // g^rr
  o[3] = Del / Sig;
  o[8] = (Del_r * Sig - Del * Sig_r) / (Sig * Sig);
  o[13] = -Del * Sig_t / (Sig * Sig);
  // g^thth
  o[4] = 1.0 / Sig;
  o[9] = -Sig_r / (Sig * Sig);
  o[14] = -Sig_t / (Sig * Sig);
}

int metric_inv(const orc_metric *m, double r, double th, double o[15]) {
  switch (m->id) {
    case 0:
      schwarzschild_inv(m->M, r, th, o);
      return 0;
    case 1:
      kerr_inv(m->M, m->a, r, th, o);
      return 0;
    case 2:  // R4-R6 evaluated literally, derivatives by complex step (analytic functions only)
      return metric_inv_complex_step(m, r, th, o);
  }
  return -1;
}

// Horizon: Schwarzschild 2M; Kerr r+ = M + sqrt(M^2-a^2) (root of eq 12);
// Manko-Novikov x = 1 <=> r = M + k (R24).
double horizon_radius(const orc_metric *m) {
  if (m->id == 0) return 2.0 * m->M;
  return m->M + std::sqrt(m->M * m->M - m->a * m->a);
}

// Prograde ISCO of Kerr (Bardeen, Press & Teukolsky 1972); Schwarzschild is a = 0.
double isco_radius(const orc_metric *m) {
  if (m->id == 2) return std::numeric_limits<double>::quiet_NaN();
  double M = m->M;
  double as = (m->id == 0 || M == 0.0) ? 0.0 : m->a / M;
  double Z1 = 1.0 + std::cbrt(1.0 - as * as) * (std::cbrt(1.0 + as) + std::cbrt(1.0 - as));
  double Z2 = std::sqrt(3.0 * as * as + Z1 * Z1);
  return M * (3.0 + Z2 - std::sqrt((3.0 - Z1) * (3.0 + Z1 + 2.0 * Z2)));
}

// Prograde circular equatorial emitter in Kerr (eq 56 solved in closed form, R19/R20):
// Omega_K = sqrt(M)/(r^{3/2} + a sqrt(M)),
// u^t = (r^{3/2} + a sqrt M)/(r^{3/4} sqrt(r^{3/2} - 3 M sqrt r + 2 a sqrt M)),
// g = (p.u_obs)/(p.u_emit) = 1/[u^t (p_t + Omega_K p_phi)]  (eq 57; p.u_obs = 1 by R12).
void kepler(const orc_metric *m, double r, double pt, double pphi, double out[3]) {
  double M = m->M, a = (m->id == 0) ? 0.0 : m->a;
  double sM = std::sqrt(M);
  double r32 = r * std::sqrt(r);
  double Om = sM / (r32 + a * sM);
  double ut = (r32 + a * sM) / (std::pow(r, 0.75) * std::sqrt(r32 - 3.0 * M * std::sqrt(r) + 2.0 * a * sM));
  out[0] = Om;
  out[1] = ut;
  out[2] = 1.0 / (ut * (pt + Om * pphi));
}

// The same emitter for any of the metrics, as the paper states it (eq 56, reading R20):
// a circular equatorial orbit has dp_r/dlambda = 0 and p_r = p_theta = 0; with p_t = -1 that is the
// quadratic  d_r g^{phi phi} p_phi^2 + 2 d_r g^{t phi} p_t p_phi + d_r g^{tt} p_t^2 = 0  in p_phi
// (the paper differentiates numerically; here the derivatives are the oracle's own d_r g^{mu nu}).
// The root with Omega > 0 is taken (the +phi direction of Omega_K = sqrt(M)/(r^{3/2} + a sqrt(M)), R19:
// co-rotating when a > 0).  Then p is
// normalised to p^2 = -1 and g = 1/[u^t (p_t + Omega p_phi)] (R19).  Returns -1 when no circular
// orbit exists at r (negative discriminant or a space-like root).
int kepler_general(const orc_metric *m, double r, double pt, double pphi, double out[3]) {
  double g[15];
  if (metric_inv(m, r, kHalfPi, g)) return -1;
  const double gtt = g[0], gtp = g[1], gpp = g[2];
  const double A = g[7], B = g[6], C = g[5];      // d_r g^{phi phi}, d_r g^{t phi}, d_r g^{tt}
  const double disc = B * B - A * C;
  if (!(disc >= 0.0)) return -1;
  double best_Om = 0.0, best_ut = 0.0;
  bool found = false;
  for (int k = 0; k < 2; ++k) {
    double pph_e = (B + (k == 0 ? 1.0 : -1.0) * std::sqrt(disc)) / A;   // p_t = -1
    double ut_raw = -gtt + gtp * pph_e;                                   // g^{t mu} p_mu
    double uph_raw = -gtp + gpp * pph_e;
    double N = -(gtt - 2.0 * gtp * pph_e + gpp * pph_e * pph_e);          // -p^2
    if (!(N > 0.0) || !(ut_raw > 0.0)) continue;
    double Om = uph_raw / ut_raw;
    if (Om > 0.0) {
      best_Om = Om;
      best_ut = ut_raw / std::sqrt(N);
      found = true;
    }
  }
  if (!found) return -1;
  out[0] = best_Om;
  out[1] = best_ut;
  out[2] = 1.0 / (best_ut * (pt + best_Om * pphi));
  return 0;
}

// ------------------------------------------------------------------------------------------
// O1: ray index -> (alpha, beta)   (R11; evaluated with individually rounded operations)
// ------------------------------------------------------------------------------------------
uint64_t splitmix_finalise(uint64_t z) {
  z += 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  z = z ^ (z >> 31);
  return z;
}

double jitter_unit(uint64_t seed, uint64_t ray, uint64_t axis) {
  uint64_t z = seed * 0x9E3779B97F4A7C15ULL + 2ULL * ray + axis;
  z = splitmix_finalise(z);
  return (double)(z >> 11) * (1.0 / 9007199254740992.0);  // 2^-53
}

void alpha_beta(const orc_camera *cam, int64_t ray, double *alpha, double *beta) {
  int64_t S = cam->supersample;
  int64_t Wt = cam->width * S;
  int64_t I = ray % Wt, J = ray / Wt;
  double jx = 0.0, jy = 0.0;
  if (cam->jitter_amp_px > 0.0) {
    jx = (2.0 * jitter_unit(cam->jitter_seed, (uint64_t)ray, 0) - 1.0) * cam->jitter_amp_px;
    jy = (2.0 * jitter_unit(cam->jitter_seed, (uint64_t)ray, 1) - 1.0) * cam->jitter_amp_px;
  }
  double X = ((double)I + 0.5) / (double)S + jx + cam->shift_x_px;
  double Y = ((double)J + 0.5) / (double)S + jy + cam->shift_y_px;
  *alpha = cam->alpha_min + X * ((cam->alpha_max - cam->alpha_min) / (double)cam->width);
  *beta = cam->beta_min + Y * ((cam->beta_max - cam->beta_min) / (double)cam->height);
}

// ------------------------------------------------------------------------------------------
// O2 + O3: pinhole in the observer's ZAMO tetrad -> covariant momentum  (R11, R12)
// Replaces P:L338-348 (eq 54-55): same content (null vector, fixed normalisation, lowered
// index), built from an orthonormal frame instead of a Euclidean screen.
// ------------------------------------------------------------------------------------------
// The paper's own camera, P:L314-348 (section 3.3.1, Fig 2-3, eq 51-55): a flat screen in Euclidean
// xyz (z = the Boyer-Lindquist axis), offset from the origin, start point and direction per pixel,
// converted to Boyer-Lindquist by inverting eq 51-53 and differentiating the inverse, made null by
// solving eq 54 for dt/dlambda, scaled so that dt/dlambda = -1, lowered with eq 55.
// Readings: the screen is centred at r_obs c_hat with c_hat the unit vector at (theta_obs, phi_obs)
// (the paper: viewing along -y, then rotating about the x axis); its axes are e_phi (alpha) and
// e_up = -e_theta (beta), the same orientation as the pinhole camera; the direction is
// -c_hat + (2f/d) (alpha e_phi + beta e_up) ("add the x and z position to the velocities,
// multiplying by a factor 2f/d").  eq 51-53 use the spin a of the metric (0 for Schwarzschild).
int initial_state_screen(const orc_metric *m, const orc_camera *cam, double alpha, double beta, double st[8]) {
  const double a = (m->id == 0) ? 0.0 : m->a;
  const double so = std::sin(cam->theta_obs), co = std::cos(cam->theta_obs);
  const double sp = std::sin(cam->phi_obs), cp = std::cos(cam->phi_obs);
  const double chat[3] = {so * cp, so * sp, co};
  const double eph[3] = {-sp, cp, 0.0};
  const double eup[3] = {-co * cp, -co * sp, so};
  const double k2 = cam->focal_2f_over_d;
  double X[3], V[3];
  for (int i = 0; i < 3; ++i) {
    X[i] = cam->r_obs * chat[i] + alpha * eph[i] + beta * eup[i];
    V[i] = -chat[i] + k2 * (alpha * eph[i] + beta * eup[i]);
  }
  // inverse of eq 51-53: r^2 is the positive root of r^4 - w r^2 - a^2 z^2 = 0, w = |X|^2 - a^2
  const double w = X[0] * X[0] + X[1] * X[1] + X[2] * X[2] - a * a;
  const double r = std::sqrt(0.5 * (w + std::sqrt(w * w + 4.0 * a * a * X[2] * X[2])));
  const double th = std::acos(X[2] / r);
  const double ph = std::atan2(X[1], X[0]);
  const double sth = std::sin(th), cth = std::cos(th), sph = std::sin(ph), cph = std::cos(ph);
  const double R = std::sqrt(r * r + a * a), Sig = r * r + a * a * cth * cth;
  // derivative of the inverse map applied to V
  const double u = V[0] * cph + V[1] * sph;
  double dph = (-V[0] * sph + V[1] * cph) / (R * sth);
  double dr = R * (r * sth * u + R * cth * V[2]) / Sig;
  double dth = (R * cth * u - r * sth * V[2]) / Sig;
  double g[5];
  if (metric_cov<double>(m, r, th, g)) return -1;
  const double gtt = g[0], gtp = g[1], gpp = g[2], grr = g[3], gthth = g[4];
  // eq 54 as a quadratic in dt: g_tt dt^2 + 2 g_tphi dphi dt + S = 0; the root with dt < 0
  const double S = grr * dr * dr + gthth * dth * dth + gpp * dph * dph;
  const double B = gtp * dph;
  const double dt = (-B + std::sqrt(B * B - gtt * S)) / gtt;
  const double sc = -1.0 / dt;  // scale so that dt/dlambda = -1
  dr *= sc;
  dth *= sc;
  dph *= sc;
  st[0] = 0.0;
  st[1] = r;
  st[2] = th;
  st[3] = ph;
  st[4] = -gtt + gtp * dph;   // eq 55 with dt = -1
  st[5] = grr * dr;
  st[6] = gthth * dth;
  st[7] = -gtp + gpp * dph;
  return 0;
}

int initial_state(const orc_metric *m, const orc_camera *cam, double alpha, double beta, double st[8]) {
  if (cam->projection == 1) return initial_state_screen(m, cam, alpha, beta, st);
  double g[5];
  if (metric_cov<double>(m, cam->r_obs, cam->theta_obs, g)) return -1;
  double gtt = g[0], gtp = g[1], gpp = g[2], grr = g[3], gthth = g[4];
  double Omega = -gtp / gpp;                              // ZAMO angular velocity
  double zeta = 1.0 / std::sqrt(-(gtt + Omega * gtp));   // u_ZAMO = zeta (d_t + Omega d_phi)
  double ro = cam->r_obs;
  double D = std::sqrt(ro * ro + alpha * alpha + beta * beta);
  double n_r = -ro / D, n_th = -beta / D, n_ph = alpha / D;  // pinhole direction, inward
  double p_r = std::sqrt(grr) * n_r;
  double p_th = std::sqrt(gthth) * n_th;
  double p_ph = std::sqrt(gpp) * n_ph;
  double p_t = 1.0 / zeta - Omega * p_ph;
  st[0] = 0.0;
  st[1] = cam->r_obs;
  st[2] = cam->theta_obs;
  st[3] = cam->phi_obs;
  st[4] = p_t;
  st[5] = p_r;
  st[6] = p_th;
  st[7] = p_ph;
  return 0;
}

// ------------------------------------------------------------------------------------------
// O4: Hamilton's equations.  y = (t, r, theta, phi, p_r, p_theta); p_t, p_phi constant
// because no metric function depends on t or phi.
//   dq^mu = g^{mu nu} p_nu                         P:L678 (eq 102)
//   dp_mu = -1/2 d_mu g^{rho sigma} p_rho p_sigma  P:L680 (eq 103) — R1; every term kept (R26)
// ------------------------------------------------------------------------------------------
struct Sys {
  const orc_metric *m;
  double pt, pphi;
};

void rhs(const Sys &S, const double y[6], double dy[6]) {
  double o[15];
  metric_inv(S.m, y[1], y[2], o);
  double pt = S.pt, pp = S.pphi, pr = y[4], pth = y[5];
  dy[0] = o[0] * pt + o[1] * pp;
  dy[1] = o[3] * pr;
  dy[2] = o[4] * pth;
  dy[3] = o[1] * pt + o[2] * pp;
  const double *dr = o + 5, *dt = o + 10;
  dy[4] = -0.5 * (dr[0] * pt * pt + 2.0 * dr[1] * pt * pp + dr[2] * pp * pp + dr[3] * pr * pr + dr[4] * pth * pth);
  dy[5] = -0.5 * (dt[0] * pt * pt + 2.0 * dt[1] * pt * pp + dt[2] * pp * pp + dt[3] * pr * pr + dt[4] * pth * pth);
}

// Landing system (R14, Henon's device): independent variable s = y[w] (w = 1: r, w = 2: theta),
// dy/ds = F(y)/F_w(y), dlambda/ds = 1/F_w(y).  z = (y[0..5], lambda).
void rhs_landing(const Sys &S, int w, const double z[7], double dz[7]) {
  double dy[6];
  rhs(S, z, dy);
  for (int i = 0; i < 6; ++i) dz[i] = dy[i] / dy[w];
  dz[6] = 1.0 / dy[w];
}

// ------------------------------------------------------------------------------------------
// O5: integrators
// ------------------------------------------------------------------------------------------

// Classical RK4 (eq 42-49 with R9), autonomous system of dimension n <= 7.
template <class F>
void rk4_step(F f, int n, const double *y, double h, double *ynew) {
  double k1[7], k2[7], k3[7], k4[7], tmp[7];
  f(y, k1);
  for (int i = 0; i < n; ++i) tmp[i] = y[i] + 0.5 * h * k1[i];
  f(tmp, k2);
  for (int i = 0; i < n; ++i) tmp[i] = y[i] + 0.5 * h * k2[i];
  f(tmp, k3);
  for (int i = 0; i < n; ++i) tmp[i] = y[i] + h * k3[i];
  f(tmp, k4);
  for (int i = 0; i < n; ++i) ynew[i] = y[i] + h / 6.0 * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
}

// Dormand & Prince (1980) 5(4) pair (R10).
const double DP_C[7] = {0.0, 1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0};
const double DP_A[7][7] = {
    {0, 0, 0, 0, 0, 0, 0},
    {1.0 / 5.0, 0, 0, 0, 0, 0, 0},
    {3.0 / 40.0, 9.0 / 40.0, 0, 0, 0, 0, 0},
    {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0, 0, 0, 0},
    {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0, 0, 0},
    {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0, 0},
    {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0, 0}};
const double DP_B[7] = {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0, 0.0};
// e = b(5th) - b*(4th)
const double DP_E[7] = {71.0 / 57600.0, 0.0, -71.0 / 16695.0, 71.0 / 1920.0, -17253.0 / 339200.0, 22.0 / 525.0, -1.0 / 40.0};

// One DP5(4) step.  k1 in (k[0]) must hold f(y).  Outputs ynew (5th order), k[6] = f(ynew),
// errvec[i] = h * sum_j e_j k_j[i].
template <class F>
void dp54_step(F f, int n, const double *y, double h, double k[7][7], double *ynew, double *errvec) {
  double tmp[7];
  for (int s = 1; s < 7; ++s) {
    for (int i = 0; i < n; ++i) {
      double acc = 0.0;
      for (int j = 0; j < s; ++j) acc += DP_A[s][j] * k[j][i];
      tmp[i] = y[i] + h * acc;
    }
    if (s == 6)
      for (int i = 0; i < n; ++i) ynew[i] = tmp[i];
    f(tmp, k[s]);
  }
  for (int i = 0; i < n; ++i) {
    double acc = 0.0;
    for (int j = 0; j < 7; ++j) acc += DP_E[j] * k[j][i];
    errvec[i] = h * acc;
  }
}

bool all_finite(const double *v, int n) {
  for (int i = 0; i < n; ++i)
    if (!std::isfinite(v[i])) return false;
  return true;
}

// R10 items 1-2: max-norm of the scaled error estimate over the six evolving components,
// sc_j = atol + rtol*max(|y_j|, |y+_j|); NaN if any term is not finite.
double error_norm(const double y[6], const double ynew[6], const double errvec[6], double rtol, double atol) {
  double err = 0.0;
  bool bad = false;
  for (int i = 0; i < 6; ++i) {
    double sc = atol + rtol * std::fmax(std::fabs(y[i]), std::fabs(ynew[i]));
    double e = std::fabs(errvec[i]) / sc;
    if (!std::isfinite(e)) bad = true;
    else if (e > err) err = e;
  }
  return bad ? std::numeric_limits<double>::quiet_NaN() : err;
}

// One landing step (R14) from state y (lambda = lam) onto y[w] = target, with the scheme's
// own formula; for the embedded pair the 5th-order solution, error estimate ignored.
void landing_step(const Sys &S, int64_t scheme, int w, const double y[6], double lam, double target,
                  double yout[6], double *lam_out) {
  double z[7], znew[7];
  for (int i = 0; i < 6; ++i) z[i] = y[i];
  z[6] = lam;
  double ds = target - y[w];
  auto f = [&](const double *zz, double *dz) { rhs_landing(S, w, zz, dz); };
  if (scheme == 2) {
    double k[7][7], errvec[7];
    f(z, k[0]);
    dp54_step(f, 7, z, ds, k, znew, errvec);
  } else {
    rk4_step(f, 7, z, ds, znew);
  }
  for (int i = 0; i < 6; ++i) yout[i] = znew[i];
  yout[w] = target;  // exact by construction (dz_w/ds = 1); remove rounding residue
  *lam_out = znew[6];
}

struct Monitors {
  double h_max, q_drift, sin_min, err_margin, Q0;
  bool have_Q0;
};

// O6 (R22, R23): sampled at every state a step is attempted from, using k1 = F(y).
void monitor(const Sys &S, const double y[6], const double k1[6], Monitors *mo) {
  double H = 0.5 * (S.pt * k1[0] + y[4] * k1[1] + y[5] * k1[2] + S.pphi * k1[3]);
  if (std::fabs(H) > mo->h_max) mo->h_max = std::fabs(H);
  double s = std::sin(y[2]), c = std::cos(y[2]);
  if (std::fabs(s) < mo->sin_min) mo->sin_min = std::fabs(s);
  if (S.m->id != 2) {
    double a = (S.m->id == 1) ? S.m->a : 0.0;
    // Carter constant, exact off shell (R23)
    double Q = y[5] * y[5] + c * c * (S.pphi * S.pphi / (s * s) - a * a * S.pt * S.pt) - 2.0 * a * a * c * c * H;
    if (!mo->have_Q0) {
      mo->Q0 = Q;
      mo->have_Q0 = true;
    }
    double d = std::fabs(Q - mo->Q0) / std::fmax(1.0, std::fabs(mo->Q0));
    if (d > mo->q_drift) mo->q_drift = d;
  }
}

struct PathSink {
  double *buf;
  int64_t cap, n;
  void push(double lam, const double y[6], double h) {
    if (!buf || n >= cap) return;
    double *p = buf + 8 * n;
    p[0] = lam;
    for (int i = 0; i < 6; ++i) p[1 + i] = y[i];
    p[7] = h;
    ++n;
  }
};

// O5-O8 for one ray.
void trace_ray(const orc_metric *m, const orc_camera *cam, const orc_cfg *cfg, double alpha, double beta,
               orc_record *rec, PathSink *path) {
  std::memset(rec, 0, sizeof(*rec));
  const double NaN = std::numeric_limits<double>::quiet_NaN();
  for (int i = 0; i < 3; ++i) rec->disk_r[i] = rec->disk_g[i] = NaN;
  rec->alpha = alpha;
  rec->beta = beta;
  double st[8];
  initial_state(m, cam, alpha, beta, st);
  Sys S;
  S.m = m;
  S.pt = st[4];
  S.pphi = st[7];
  double y[6] = {st[0], st[1], st[2], st[3], st[5], st[6]};
  double lam = 0.0;
  const int64_t scheme = cfg->scheme;
  const double r_cap = horizon_radius(m) * (1.0 + cfg->eps_capture);
  const double r_esc = cfg->r_escape;
  const bool disk_on = cfg->max_crossings > 0;
  const bool ring_on = cfg->ring_half_angle > 0.0;
  const double ring_d = cfg->ring_half_angle;
  double r_in = cfg->disk_r_in, r_out = cfg->disk_r_out;
  if ((disk_on || ring_on) && r_in <= 0.0) r_in = isco_radius(m);
  Monitors mo;
  mo.h_max = 0.0;
  mo.q_drift = 0.0;
  mo.sin_min = std::numeric_limits<double>::infinity();
  mo.err_margin = std::numeric_limits<double>::infinity();
  mo.Q0 = 0.0;
  mo.have_Q0 = false;
  int64_t n_acc = 0, n_rej = 0, n_cross = 0, n_rec = 0, n_land = 0;
  int64_t status = -1;
  auto f = [&](const double *yy, double *dy) { rhs(S, yy, dy); };

  double h = (scheme == 2) ? cfg->h_cap_rel * st[1] : 0.0;  // R10 item 4 (st[1] = r_obs for the pinhole)
  double k[7][7];
  if (scheme == 2) f(y, k[0]);
  if (path) path->push(lam, y, h);

  for (;;) {
    if (n_acc + n_rej >= cfg->max_steps) {  // R18
      status = 2;
      break;
    }
    if (cfg->lambda_max > 0.0 && lam >= cfg->lambda_max) {
      status = 2;
      break;
    }
    double ynew[6], hnext = 0.0;
    bool stage_captured = false;
    if (scheme == 2) {
      if (h < 1e-14 * std::fmax(1.0, std::fabs(lam))) {
        status = 4;
        break;
      }
      monitor(S, y, k[0], &mo);
      double errvec[7];
      dp54_step(f, 6, y, h, k, ynew, errvec);
      // R10 items 1-3: max-norm of the scaled error over the six evolving components
      double err = error_norm(y, ynew, errvec, cfg->rtol, cfg->atol);
      if (!std::isfinite(err) || !all_finite(ynew, 6)) {
        ++n_rej;
        h *= 0.2;
        continue;
      }
      double margin = std::fabs(err - 1.0);
      if (margin < mo.err_margin) mo.err_margin = margin;
      double fac = (err == 0.0) ? 5.0 : 0.9 * std::pow(err, -0.2);
      if (err > 1.0) {
        ++n_rej;
        h *= std::fmax(0.2, fac);
        continue;
      }
      ++n_acc;
      hnext = std::fmin(h * std::fmin(5.0, std::fmax(0.2, fac)), cfg->h_cap_rel * ynew[1]);
    } else {
      h = (scheme == 0) ? cfg->h : cfg->h_rel * y[1];  // R17
      f(y, k[0]);
      monitor(S, y, k[0], &mo);
      // Classical RK4 (eq 42-49, R9) written out so that every state the equations are
      // evaluated at passes the capture test first (R31): a fixed step taken from just outside
      // the capture radius would otherwise evaluate the metric on or inside the horizon, where
      // the coordinates are singular (P:L394 notes the artefact).
      double y2[6], y3[6], y4[6];
      for (int i = 0; i < 6; ++i) y2[i] = y[i] + 0.5 * h * k[0][i];
      stage_captured = y2[1] < r_cap;
      if (!stage_captured) {
        f(y2, k[1]);
        for (int i = 0; i < 6; ++i) y3[i] = y[i] + 0.5 * h * k[1][i];
        stage_captured = y3[1] < r_cap;
      }
      if (!stage_captured) {
        f(y3, k[2]);
        for (int i = 0; i < 6; ++i) y4[i] = y[i] + h * k[2][i];
        stage_captured = y4[1] < r_cap;
      }
      if (!stage_captured) {
        f(y4, k[3]);
        for (int i = 0; i < 6; ++i)
          ynew[i] = y[i] + h / 6.0 * (k[0][i] + 2.0 * k[1][i] + 2.0 * k[2][i] + k[3][i]);
        if (!all_finite(ynew, 6)) {
          status = 3;
          break;
        }
      }
      ++n_acc;
    }
    // O8: termination on the accepted step, landing from the state before it (R14)
    if (stage_captured || ynew[1] > r_esc || ynew[1] < r_cap) {
      bool esc = !stage_captured && ynew[1] > r_esc;
      double target = esc ? r_esc : r_cap;
      status = esc ? 0 : 1;
      double yl[6], laml;
      landing_step(S, scheme, 1, y, lam, target, yl, &laml);
      ++n_land;
      for (int i = 0; i < 6; ++i) y[i] = yl[i];
      lam = laml;
      break;
    }
    // Solid ring ("collision is based on the ray propagating to a point inside volume of the
    // object"; reading R39).  Volume: r_in <= r <= r_out, |theta - pi/2| <= d, a box in (r, theta).
    // An accepted, non-terminal step y_n -> y_{n+1} (y_n outside the volume) can meet it only if every
    // coordinate that starts outside its interval ENTERS it during the step (ends inside it or beyond
    // it).  Then the entry point is LOCATED with the landing step of R14 from y_n, on the face of each such
    // coordinate on y_n's side: the theta-face first — a hit if the landed radius is in range — else the
    // radial face — a hit if the landed theta is inside the slab.  (For a ray that enters the box, the
    // later of the two face crossings is the entry and only there is the other coordinate in range.)
    // This contains the paper's test (y_{n+1} inside) and does not depend on the step size for a slab
    // or a corner crossed within one step.
    if (ring_on) {
      const double un = y[2] - kHalfPi, un1 = ynew[2] - kHalfPi;
      const bool th_out = std::fabs(un) > ring_d;
      const bool r_out_n = !(y[1] >= r_in && y[1] <= r_out);
      const bool th_enters = std::fabs(un1) <= ring_d || un * un1 < 0.0;
      const bool r_enters = (ynew[1] >= r_in && ynew[1] <= r_out) || (y[1] < r_in) != (ynew[1] < r_in);
      double yl[6], laml;
      bool hit = false;
      if ((th_out || r_out_n) && (!th_out || th_enters) && (!r_out_n || r_enters)) {
        if (th_out) {
          landing_step(S, scheme, 2, y, lam, kHalfPi + (un > 0.0 ? ring_d : -ring_d), yl, &laml);
          ++n_land;
          hit = yl[1] >= r_in && yl[1] <= r_out;
        }
        if (!hit && r_out_n) {
          landing_step(S, scheme, 1, y, lam, (y[1] < r_in) ? r_in : r_out, yl, &laml);
          ++n_land;
          hit = std::fabs(yl[2] - kHalfPi) <= ring_d;
        }
      }
      if (hit) {
        double kp[3] = {NaN, NaN, NaN};
        if (m->id == 2) kepler_general(m, yl[1], S.pt, S.pphi, kp);
        else kepler(m, yl[1], S.pt, S.pphi, kp);
        rec->disk_r[0] = yl[1];
        rec->disk_g[0] = kp[2];
        n_rec = 1;
        for (int i = 0; i < 6; ++i) y[i] = yl[i];
        lam = laml;
        status = 5;
        break;
      }
    }
    // O7: equator crossing on an accepted, non-terminal step (R19)
    if ((y[2] - kHalfPi) * (ynew[2] - kHalfPi) < 0.0) {
      ++n_cross;
      if (disk_on && n_rec < cfg->max_crossings) {
        double yl[6], laml;
        landing_step(S, scheme, 2, y, lam, kHalfPi, yl, &laml);
        ++n_land;
        double rc = yl[1];
        if (rc >= r_in && rc <= r_out) {
          double kp[3] = {NaN, NaN, NaN};
          if (m->id == 2) kepler_general(m, rc, S.pt, S.pphi, kp);   // no circular orbit there: g = NaN
          else kepler(m, rc, S.pt, S.pphi, kp);
          rec->disk_r[n_rec] = rc;
          rec->disk_g[n_rec] = kp[2];
          ++n_rec;
        }
      }
    }
    for (int i = 0; i < 6; ++i) y[i] = ynew[i];
    lam += h;
    if (scheme == 2) {
      for (int i = 0; i < 6; ++i) k[0][i] = k[6][i];  // FSAL
      h = hnext;
    }
    if (path) path->push(lam, y, h);
  }
  if (path) path->push(lam, y, h);

  rec->status = status;
  rec->n_accepted = n_acc;
  rec->n_rejected = n_rej;
  rec->n_equator_crossings = n_cross;
  rec->n_disk_recorded = n_rec;
  // evaluations the method needs: DP5(4) 1 + 6/attempt + 5/landing (k1 reused);
  // RK4 4/step + 3/landing
  rec->n_rhs = (scheme == 2) ? 1 + 6 * (n_acc + n_rej) + 5 * n_land : 4 * n_acc + 3 * n_land;
  rec->t = y[0];
  rec->r = y[1];
  rec->theta = y[2];
  rec->phi = y[3];
  rec->p_r = y[4];
  rec->p_theta = y[5];
  rec->p_t = S.pt;
  rec->p_phi = S.pphi;
  rec->lambda = lam;
  rec->h_max = mo.h_max;
  rec->q_drift = mo.q_drift;
  rec->sin_theta_min = mo.sin_min;
  rec->err_margin = mo.err_margin;
}

bool valid_metric(const orc_metric *m) {
  if (!m) return false;
  if (m->id < 0 || m->id > 2) return false;
  if (m->id == 0) return m->M >= 0.0;
  if (!(m->M > 0.0) || !(std::fabs(m->a) < m->M)) return false;
  if (m->id == 2 && m->a == 0.0) return false;  // eq 23 divides by S/M
  return true;
}

}  // namespace

extern "C" {

void orc_alpha_beta(const orc_camera *cam, int64_t ray, double *alpha, double *beta) {
  alpha_beta(cam, ray, alpha, beta);
}

int orc_metric_cov(const orc_metric *m, double r, double theta, double *out5) {
  if (!valid_metric(m)) return -1;
  return metric_cov<double>(m, r, theta, out5);
}

int orc_metric_inv(const orc_metric *m, double r, double theta, double *out15) {
  if (!valid_metric(m)) return -1;
  return metric_inv(m, r, theta, out15);
}

int orc_metric_inv_complex_step(const orc_metric *m, double r, double theta, double *out15) {
  if (!valid_metric(m)) return -1;
  return metric_inv_complex_step(m, r, theta, out15);
}

int orc_mn_potentials(const orc_metric *m, double r, double theta, double *out10) {
  if (!valid_metric(m) || m->id != 2) return -1;
  MNConst c = mn_constants(m->M, m->a, m->q);
  MNPot<double> o = mn_potentials<double>(c, r, theta);
  out10[0] = o.f;
  out10[1] = o.omega;
  out10[2] = o.e2gamma;
  out10[3] = o.A;
  out10[4] = o.B;
  out10[5] = o.C;
  out10[6] = o.afr;
  out10[7] = o.bfr;
  out10[8] = o.psi;
  out10[9] = o.gammap;
  return 0;
}

int orc_initial_state(const orc_metric *m, const orc_camera *cam, double alpha, double beta, double *state8) {
  if (!valid_metric(m)) return -1;
  return initial_state(m, cam, alpha, beta, state8);
}

int orc_rhs(const orc_metric *m, const double *st, double *rhs6) {
  if (!valid_metric(m)) return -1;
  Sys S;
  S.m = m;
  S.pt = st[4];
  S.pphi = st[7];
  double y[6] = {st[0], st[1], st[2], st[3], st[5], st[6]};
  rhs(S, y, rhs6);
  return 0;
}

int orc_radii(const orc_metric *m, double *r_horizon, double *r_isco) {
  if (!valid_metric(m)) return -1;
  *r_horizon = horizon_radius(m);
  *r_isco = isco_radius(m);
  return 0;
}

int orc_kepler(const orc_metric *m, double r, double p_t, double p_phi, double *out3) {
  if (!valid_metric(m) || m->id == 2) return -1;
  kepler(m, r, p_t, p_phi, out3);
  return 0;
}

int orc_kepler_general(const orc_metric *m, double r, double p_t, double p_phi, double *out3) {
  if (!valid_metric(m)) return -1;
  return kepler_general(m, r, p_t, p_phi, out3);
}

void orc_dp54_tableau(double *c7, double *a49, double *b7, double *e7) {
  for (int i = 0; i < 7; ++i) {
    c7[i] = DP_C[i];
    b7[i] = DP_B[i];
    e7[i] = DP_E[i];
    for (int j = 0; j < 7; ++j) a49[7 * i + j] = DP_A[i][j];
  }
}

int orc_single_step(const orc_metric *m, int64_t scheme, const double *st, double h, double rtol, double atol,
                    double *out_state8, double *err_out) {
  if (!valid_metric(m)) return -1;
  Sys S;
  S.m = m;
  S.pt = st[4];
  S.pphi = st[7];
  double y[6] = {st[0], st[1], st[2], st[3], st[5], st[6]}, ynew[6];
  auto f = [&](const double *yy, double *dy) { rhs(S, yy, dy); };
  double err = 0.0;
  if (scheme == 2) {
    double k[7][7], errvec[7];
    f(y, k[0]);
    dp54_step(f, 6, y, h, k, ynew, errvec);
    err = error_norm(y, ynew, errvec, rtol, atol);
  } else {
    rk4_step(f, 6, y, h, ynew);
  }
  out_state8[0] = ynew[0];
  out_state8[1] = ynew[1];
  out_state8[2] = ynew[2];
  out_state8[3] = ynew[3];
  out_state8[4] = st[4];
  out_state8[5] = ynew[4];
  out_state8[6] = ynew[5];
  out_state8[7] = st[7];
  *err_out = err;
  return 0;
}

static int valid_run(const orc_metric *m, const orc_camera *cam, const orc_cfg *cfg) {
  if (!valid_metric(m) || !cam || !cfg) return 0;
  if (cfg->scheme < 0 || cfg->scheme > 2) return 0;
  if (cfg->max_crossings < 0 || cfg->max_crossings > 3) return 0;
  if (!(cfg->ring_half_angle >= 0.0) || cfg->ring_half_angle >= 1.5) return 0;
  if (cfg->ring_half_angle > 0.0 && (cfg->max_crossings > 0 || !(cfg->disk_r_out >= cfg->disk_r_in)))
    return 0;   // the ring replaces the thin disk
  if (cfg->ring_half_angle > 0.0 && m->id == 2 && !(cfg->disk_r_in > 0.0)) return 0;
  if (cfg->max_crossings > 0 && m->id == 2 && !(cfg->disk_r_in > 0.0)) return 0;  // no ISCO formula for Manko-Novikov
  if (cam->width <= 0 || cam->height <= 0 || cam->supersample <= 0) return 0;
  return 1;
}

int orc_trace(const orc_metric *m, const orc_camera *cam, const orc_cfg *cfg, int64_t ray_begin, int64_t ray_count,
              int64_t ray_stride, orc_record *out, int n_threads) {
  if (!valid_run(m, cam, cfg) || !out || ray_count < 0 || ray_stride < 1) return -1;
  int used = 1;
#ifdef _OPENMP
  if (n_threads <= 0) n_threads = omp_get_max_threads();
  used = n_threads;
#pragma omp parallel for schedule(dynamic, 16) num_threads(n_threads)
#endif
  for (int64_t kk = 0; kk < ray_count; ++kk) {
    int64_t ray = ray_begin + kk * ray_stride;
    double al, be;
    alpha_beta(cam, ray, &al, &be);
    trace_ray(m, cam, cfg, al, be, &out[kk], nullptr);
  }
  return used;
}

int orc_trace_one(const orc_metric *m, const orc_camera *cam, const orc_cfg *cfg, double alpha, double beta,
                  orc_record *out, double *path, int64_t n_path_max, int64_t *n_path) {
  if (!valid_run(m, cam, cfg) || !out) return -1;
  PathSink sink;
  sink.buf = path;
  sink.cap = n_path_max;
  sink.n = 0;
  trace_ray(m, cam, cfg, alpha, beta, out, path ? &sink : nullptr);
  if (n_path) *n_path = sink.n;
  return 0;
}

// Orbits from explicit initial states (the time-like test orbits of section 3.2.1 are
// the same equations with H = -1/2; neighbouring null orbits).  See gp_oracle.h.
int orc_integrate_orbits(const orc_metric *m, const orc_orbit_cfg *cfg, const double *states8, int64_t n,
                         double *samples, int64_t *status, int64_t *n_steps) {
  if (!m || !cfg || !states8 || !samples || n < 0 || cfg->n_samples < 1) return -1;
  if (!(cfg->rtol > 0.0) || !(cfg->atol >= 0.0) || !(cfg->h0 > 0.0) || !(cfg->h_max > 0.0) ||
      !(cfg->lambda_end > 0.0))
    return -1;
  const double r_cap = horizon_radius(m) * (1.0 + cfg->eps_capture);
  const double NaN = std::numeric_limits<double>::quiet_NaN();
  const int64_t K = cfg->n_samples;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t i = 0; i < n; ++i) {
    const double *st = states8 + 8 * i;
    double *out = samples + 8 * K * i;
    for (int64_t j = 0; j < 8 * K; ++j) out[j] = NaN;
    Sys S;
    S.m = m;
    S.pt = st[4];
    S.pphi = st[7];
    auto f = [&](const double *yy, double *dy) { rhs(S, yy, dy); };
    double y[6] = {st[0], st[1], st[2], st[3], st[5], st[6]};
    // "Integrate to lambda_1, sample; integrate on to lambda_2, sample; ..." (gp_oracle.h): an outer loop over
    // the sample times and, for each, the adaptive loop of R10 run until the affine parameter EQUALS the
    // sample time.  `proposal` is the controller's current step suggestion; an attempt takes the smallest of
    // the proposal, h_max and the distance left to the sample time; when it is the distance that binds, the
    // attempt "arrives": lambda is set to the sample time itself and the proposal is not allowed to shrink
    // because of the shortened step (it keeps the larger of its old value and the new suggestion).
    double lam = 0.0, proposal = cfg->h0;
    double k[7][7];
    f(y, k[0]);
    int64_t steps = 0, stat = 0;
    for (int64_t sample = 0; sample < K && stat == 0; ++sample) {
      const double t_sample = (double)(sample + 1) * cfg->lambda_end / (double)K;
      while (lam != t_sample) {
        if (steps >= cfg->max_steps) { stat = 2; break; }
        if (proposal < 1e-14 * std::fmax(1.0, std::fabs(lam))) { stat = 4; break; }
        const double left = t_sample - lam;
        double take = std::fmin(proposal, cfg->h_max);
        const bool arrives = take >= left;
        if (arrives) take = left;
        double ynew[6], errvec[7];
        dp54_step(f, 6, y, take, k, ynew, errvec);
        ++steps;
        const double err = error_norm(y, ynew, errvec, cfg->rtol, cfg->atol);
        if (!std::isfinite(err) || !all_finite(ynew, 6)) {   // R10 item 2
          proposal = 0.2 * take;
          continue;
        }
        const double fac = (err == 0.0) ? 5.0 : 0.9 * std::pow(err, -0.2);
        if (err > 1.0) {                                     // R10 item 3, rejected
          proposal = take * std::fmax(0.2, fac);
          continue;
        }
        const double suggestion = take * std::fmin(5.0, std::fmax(0.2, fac));
        proposal = arrives ? std::fmax(proposal, suggestion) : suggestion;
        for (int c = 0; c < 6; ++c) y[c] = ynew[c];
        for (int c = 0; c < 6; ++c) k[0][c] = k[6][c];       // FSAL
        lam = arrives ? t_sample : lam + take;
        if (y[1] < r_cap) { stat = 1; break; }
      }
      if (stat != 0) break;
      // the sample: state, 2H = p_mu dq^mu/dlambda from the slopes at the new state, lambda
      double *o = out + 8 * sample;
      o[0] = y[0]; o[1] = y[1]; o[2] = y[2]; o[3] = y[3]; o[4] = y[4]; o[5] = y[5];
      o[6] = S.pt * k[0][0] + y[4] * k[0][1] + y[5] * k[0][2] + S.pphi * k[0][3];
      o[7] = lam;
    }
    status[i] = stat;
    n_steps[i] = steps;
  }
  return 0;
}

}  // extern "C"
