// gp_metric.cuh — per-metric device functions: Hamilton's equations (SURVEY.md section 8 rows
// a4 + a5), the covariant metric at the observer (row a3, host side) and the 15-number
// inverse-metric table behind gp_eval_metric.
//
//   H = 1/2 g^{mu nu} p_mu p_nu                                   PAPER.md L116 (eq 3)
//   dq^mu/dlambda = g^{mu nu} p_nu                                PAPER.md L678 (eq 102)
//   dp_mu/dlambda = -1/2 d_mu g^{rho sigma} p_rho p_sigma          PAPER.md L680 (eq 103), reading R1
//
// Schwarzschild (eq 8) and Kerr in Boyer-Lindquist coordinates (PAPER.md
// L147-159, eq 9-14, readings R2/R3) use closed forms; Manko-Novikov (PAPER.md L181-230,
// eq 20-39, readings R4-R8) differentiates the Hamiltonian with forward-mode dual numbers.
// All three metrics depend on (r, theta) only, so p_t and p_phi are constants of the ray and
// every function here takes them as parameters.
#ifndef GP_METRIC_CUH_
#define GP_METRIC_CUH_

#include "gp_dual.cuh"

namespace gp {

enum { METRIC_SCHW = 0, METRIC_KERR = 1, METRIC_MN = 2 };

// Constants of the spacetime, derived once on the host (gp_api.cu).
struct MetricConst {
  double M, a, q;
  double a2;        // a^2
  double m2M;       // -2M
  double r_horizon; // 2M | M + sqrt(M^2-a^2) | M + k
  // Manko-Novikov, PAPER.md L192-196 (eq 23-25), reading R7
  double mn_alpha;  // (-M + sqrt(M^2-a^2))/a
  double mn_k;      // M (1-alpha^2)/(1+alpha^2)
  double mn_inv_k;
  double mn_beta;   // q M^3/k^3
  double mn_w0;     // 4 k alpha/(1-alpha^2)          (eq 27, constant part of omega)
  double mn_e0;     // k^2/(1-alpha^2)^2              (eq 28 with the ln term cancelled, see mn_core)
};

// Derivatives of (t, r, theta, phi, p_r, p_theta) with respect to the affine parameter, plus the
// by-products the monitors want: sin, cos of theta and 2H.  T is the
// arithmetic type: double (required), float (the cfg.precision = 1 variant).
template <class T>
struct RhsT {
  T dt, dr, dth, dph, dpr, dpth;
  T s, c, H2;
  T is;  // 1/sin(theta) (Schwarzschild, Kerr; 0 for Manko-Novikov)
  T pw;  // Kerr: p_th^2 + W^2, W = p_ph/s + a s p_t (a by-product the Carter monitor reuses)
};
typedef RhsT<double> Rhs;

// ---- Schwarzschild --------------------------------------------------------------------------
// 2H = -p_t^2/F + F p_r^2 + p_th^2/r^2 + p_ph^2/(r^2 s^2),  F = 1 - 2M/r   (eq 8 inverted)
template <class T, bool GIVEN_SC = false>
GP_HD void rhs_schwarzschild(const MetricConst &mc, T pt, T pph, T r, T th, T pr, T pth, RhsT<T> &o,
                             T s_in = T(0), T c_in = T(0)) {
  T s, c;
  if (GIVEN_SC) {
    s = s_in;
    c = c_in;
  } else {
    fsincos(th, &s, &c);
  }
  const T M = (T)mc.M;
  T ir = frcp(r);
  T ir2 = ir * ir;
  T F = T(1) - T(2) * M * ir;
  T iF = frcp(F);
  T is = frcp(s);
  T is2 = is * is;
  T Fr = T(2) * M * ir2;              // dF/dr
  T gpp = ir2 * is2;                  // g^{phi phi}
  T pt_iF = pt * iF;
  o.dt = -pt_iF;
  o.dr = F * pr;
  o.dth = pth * ir2;
  o.dph = pph * gpp;
  T ang = pth * pth + pph * pph * is2; // p_th^2 + p_ph^2/s^2
  o.dpr = T(-0.5) * Fr * (pt_iF * pt_iF + pr * pr) + ang * ir2 * ir;
  o.dpth = c * is * pph * pph * gpp;
  o.H2 = -pt * pt_iF + F * pr * pr + ang * ir2;
  o.s = s;
  o.c = c;
  o.is = is;
}

// ---- Kerr -----------------------------------------------------------------------------------
// Compact form of the inverse Boyer-Lindquist metric (eq 9-13 inverted):
//   Sigma = r^2 + a^2 c^2, Delta = r^2 - 2Mr + a^2,
//   P = (r^2+a^2) p_t + a p_ph,  W = p_ph/s + a s p_t,
//   N = Delta p_r^2 + p_th^2 + W^2 - P^2/Delta,   2H = N/Sigma.
// Written out operation by operation (half-derivatives, shared products, explicit fma): 53 FP64
// instructions beside the sincos and the reciprocal, against 61 for the textbook arrangement — the
// FP64 pipe is the bound, so the operation count is the run time.
// SCALED: the six derivatives come out multiplied by hs, the step of the attempt, at the cost of ONE
// extra multiplication (hs / Sigma replaces 1 / Sigma in their last product); the Runge-Kutta sums
// then need no multiplication by the step (gp_trace_dp54.cuh).  The by-products (s, c, H2, is) are
// never scaled.
// GIVEN_SC: sin and cos of theta are supplied by the caller (s_in, c_in) and th is not read.
template <class T, bool SCALED = false, bool GIVEN_SC = false>
GP_HD void rhs_kerr(const MetricConst &mc, T pt, T pph, T r, T th, T pr, T pth, RhsT<T> &o, T hs = T(1),
                    T s_in = T(0), T c_in = T(0)) {
  T s, c;
  if (GIVEN_SC) {
    s = s_in;
    c = c_in;
  } else {
    fsincos(th, &s, &c);
  }
  const T a = (T)mc.a, a2 = (T)mc.a2;
  T r2 = r * r;
  T rr = r2 + a2;
  T a2c = a2 * c;
  T Sig = ffma(a2c, c, r2);
  T Del = ffma((T)mc.m2M, r, rr);
  // one reciprocal for the three denominators Sigma, Delta, s
  T SD = Sig * Del;
  T inv = frcp(SD * s);
  T is = inv * SD;
  T t1 = inv * s;
  T iSig = t1 * Del;
  T iDel = t1 * Sig;
  T as = a * s;
  T W = ffma(pph, is, as * pt);
  T P = ffma(rr, pt, a * pph);
  T PiD = P * iDel;
  T pr2 = pr * pr;
  T pw = ffma(W, W, pth * pth);
  T N = ffma(-P, PiD, ffma(Del, pr2, pw));
  T H2 = N * iSig;
  const T hS = SCALED ? hs * iSig : iSig;
  o.dt = ffma(-rr, PiD, as * W) * hS;
  o.dph = ffma(-a, PiD, W * is) * hS;
  o.dr = (pr * hS) * Del;
  o.dth = pth * hS;
  // dp_r = -(1/2 d_r N - r 2H)/Sigma,  1/2 d_r N = (r-M)(p_r^2 + (P/Delta)^2) - 2 r p_t P/Delta
  T halfNr = ffma(T(-2), (r * pt) * PiD, (r - (T)mc.M) * ffma(PiD, PiD, pr2));
  o.dpr = ffma(r, H2, -halfNr) * hS;
  // dp_th = -(1/2 d_th N + a^2 s c 2H)/Sigma,  1/2 d_th N = W c (a p_t - p_ph/s^2)
  T halfNth = (W * c) * ffma(-(pph * is), is, a * pt);
  o.dpth = -ffma(a2c * s, H2, halfNth) * hS;
  o.H2 = H2;
  o.s = s;
  o.c = c;
  o.is = is;
  o.pw = pw;
}

// ---- Manko-Novikov --------------------------------------------------------------------------
// Potentials f, omega and E = e^{2 gamma} rho^2 in prolate spheroidal x, y (eq 21-39).
// T is double (host: observer's metric) or Dual2 (device: derivatives along x and y).
// The 1/2 ln[(x^2-1)/(x^2-y^2)] term of gamma' (eq 33, R6) cancels exactly against
// rho^2/(x^2-1) in e^{2 gamma} rho^2 = e^{2 gamma'} A k^2 (x^2-y^2) / ((x^2-1)(1-alpha^2)^2),
// leaving E = k^2 A e^{2 gt}/(1-alpha^2)^2 with gt = gamma' minus that term: no log and no
// division by x^2-1.
template <class T> struct scalar_of { typedef T type; };
template <class S> struct scalar_of<Dual2T<S> > { typedef S type; };

template <class T>
struct MNCore {
  T f, omega, E;
  T iF, fE;   // 1/f and f/E as Hamilton's equations use them (see the end of mn_core)
};

template <class T>
GP_HD MNCore<T> mn_core(const MetricConst &mc, const T &x, const T &y) {
  const double al = mc.mn_alpha, be = mc.mn_beta, k = mc.mn_k;
  T x2 = sqr(x), y2 = sqr(y);
  T R2 = x2 + y2 - 1.0;            // eq 36
  // FP64: 1/R by one reciprocal square root, and below 1/f from the reciprocals omega needs anyway, so that no
  // reciprocal waits for f (config 4 -2 to -4 %).  The FP32 instantiations keep the forms their
  // tolerance was established with (reciprocal then square root, reciprocal of f).
  constexpr bool kShortChains = sizeof(typename scalar_of<T>::type) == 8;
  T iR, iR2;
  if (kShortChains) {
    iR = drsqrt(R2);               // 1/R
    iR2 = sqr(iR);
  } else {
    iR2 = recip(R2);
    iR = dsqrt(iR2);
  }
  T u = x * y * iR;                // eq 37
  T u2 = sqr(u);
  T P2 = 1.5 * u2 - 0.5;           // Legendre P_2
  T P3 = (2.5 * u2 - 1.5) * u;     // Legendre P_3
  T iR3 = iR2 * iR;
  T T0 = iR, T1 = u * iR2, T2 = P2 * iR3;  // P_l / R^{l+1}
  T psi = be * T2;                 // eq 32
  T Sa = (x - y) * (T0 + T1 + T2);         // sum in eq 34
  T Sb = (x + y) * (T1 - T0 - T2);         // sum in eq 35: (-1)^{3-l}
  T afr = -al * dexp(-2.0 * be * (Sa - 1.0));   // eq 34
  T bfr = al * dexp(2.0 * be * (1.0 + Sb));     // eq 35
  // gt: eq 33 without the log term; the l-sum there equals Sa - Sb
  T gt = (1.5 * be * be) * sqr(iR3) * (sqr(P3) - sqr(P2)) + be * (Sa - Sb - 2.0);
  T ab = afr * bfr;
  T bma = bfr - afr;
  T opab = 1.0 + ab;
  T xm = x2 - 1.0, ym = 1.0 - y2;
  T A = xm * sqr(opab) - ym * sqr(bma);                               // eq 29
  T B = sqr((x + 1.0) + (x - 1.0) * ab) + sqr((1.0 + y) * afr + (1.0 - y) * bfr);  // eq 30 (R5)
  T C = xm * opab * (bma - y * (afr + bfr)) + ym * bma * (opab + x * (1.0 - ab));  // eq 31
  T e2psi = dexp(2.0 * psi);
  MNCore<T> o;
  if (kShortChains) {
    T iB = recip(B);
    T g = recip(A) * recip(e2psi);                                    // 1/(A e^{2 psi}), shared by omega and 1/f
    o.f = e2psi * A * iB;                                             // eq 26
    o.omega = (2.0 * k) * C * g - mc.mn_w0;                           // eq 27
    o.iF = B * g;
  } else {
    T iA = recip(A);
    o.f = e2psi * A * recip(B);                                       // eq 26
    o.omega = (2.0 * k) * C * iA * recip(e2psi) - mc.mn_w0;           // eq 27
    o.iF = recip(o.f);
  }
  o.E = mc.mn_e0 * A * dexp(2.0 * gt);                                // eq 28 x rho^2
  // f/E keeps its reciprocal of E: the form in which A cancels, e^{2 psi - 2 gt}/(e0 B), stays finite where this
  // product overflows, and that changes how rays that step onto the singular horizon end.
  o.fE = o.f * recip(o.E);
  return o;
}

// 2H = -p_t^2/f + f (p_ph + omega p_t)^2/(Delta s^2) + f (Delta p_r^2 + p_th^2)/E,
// Delta = k^2 (x^2-1) (eq 22), from the line element eq 20 (R4).
template <class T>
GP_HD void rhs_manko_novikov(const MetricConst &mc, T pt, T pph, T r, T th, T pr, T pth, RhsT<T> &o) {
  typedef Dual2T<T> D;
  T s, c;
  fsincos(th, &s, &c);
  const T k = (T)mc.mn_k, ik = (T)mc.mn_inv_k;
  D x((r - (T)mc.M) * ik, T(1), T(0));
  D y(c, T(0), T(1));
  MNCore<D> m = mn_core<D>(mc, x, y);
  D Del = (k * k) * (sqr(x) - T(1));
  D s2(s * s, T(0), T(-2) * c);          // sin^2 = 1 - y^2
  D iDs = recip(Del * s2);
  const D &iF = m.iF;
  D L = pph + m.omega * pt;               // p_ph + omega p_t
  D fL = m.f * L * iDs;                   // = dphi/dlambda
  const D &fE = m.fE;                     // g^{th th}
  D K = Del * (pr * pr) + pth * pth;
  D H2 = fL * L + fE * K - (pt * pt) * iF;
  o.dt = -pt * iF.v + m.omega.v * fL.v;
  o.dph = fL.v;
  o.dr = fE.v * Del.v * pr;
  o.dth = fE.v * pth;
  o.dpr = T(-0.5) * H2.dx * ik;           // d/dr = (1/k) d/dx
  o.dpth = T(0.5) * H2.dy * s;            // d/dtheta = -sin(theta) d/dy
  o.H2 = H2.v;
  o.s = s;
  o.c = c;
  o.is = T(0);
}

#if defined(__CUDACC__)
// The Manko-Novikov evaluation is ~1000 instructions; inlined seven times it made trace_dp54<MN> 106 KB
// of code and instruction fetch its largest stall (ncu: no_instruction 1.5 per issue).  One
// out-of-line copy keeps that kernel inside the instruction cache: measured +9 % on the DP5(4) kernel
// and -4 % on the four-stage RK4 kernel, which therefore keeps the inlined form (OUTLINE_MN = false).
template <class T>
__device__ __noinline__ RhsT<T> rhs_manko_novikov_call(const MetricConst &mc, T pt, T pph, T r, T th, T pr, T pth) {
  RhsT<T> o;
  rhs_manko_novikov<T>(mc, pt, pph, r, th, pr, pth, o);
  o.pw = T(0);
  return o;   // by value: the ten results come back in registers, not through the caller's stack frame
}
#endif

template <int METRIC, bool OUTLINE_MN = false, class T>
GP_HD void rhs_eval(const MetricConst &mc, T pt, T pph, T r, T th, T pr, T pth, RhsT<T> &o) {
  if (METRIC == METRIC_SCHW) rhs_schwarzschild<T>(mc, pt, pph, r, th, pr, pth, o);
  else if (METRIC == METRIC_KERR) rhs_kerr<T>(mc, pt, pph, r, th, pr, pth, o);
  else {
#if defined(__CUDA_ARCH__)
    if (OUTLINE_MN) o = rhs_manko_novikov_call<T>(mc, pt, pph, r, th, pr, pth);
    else rhs_manko_novikov<T>(mc, pt, pph, r, th, pr, pth, o);
#else
    rhs_manko_novikov<T>(mc, pt, pph, r, th, pr, pth, o);
#endif
  }
}

// rhs_eval_scaled: the six derivatives multiplied by hs (see rhs_kerr); Schwarzschild and
// Manko-Novikov scale the results afterwards (their cost is elsewhere).
template <int METRIC, bool OUTLINE_MN = false, class T>
GP_HD void rhs_eval_scaled(const MetricConst &mc, T pt, T pph, T r, T th, T pr, T pth, T hs, RhsT<T> &o) {
  if (METRIC == METRIC_KERR) {
    rhs_kerr<T, true>(mc, pt, pph, r, th, pr, pth, o, hs);
  } else {
    rhs_eval<METRIC, OUTLINE_MN, T>(mc, pt, pph, r, th, pr, pth, o);
    o.dt *= hs; o.dr *= hs; o.dth *= hs; o.dph *= hs; o.dpr *= hs; o.dpth *= hs;
  }
}

// The same with sin and cos of theta supplied by the caller (Schwarzschild, Kerr; gp_trace_dp54.cuh
// obtains them for the stage angles by the addition theorems).
template <int METRIC, class T>
GP_HD void rhs_eval_scaled_sc(const MetricConst &mc, T pt, T pph, T r, T s, T c, T pr, T pth, T hs, RhsT<T> &o) {
  if (METRIC == METRIC_KERR) {
    rhs_kerr<T, true, true>(mc, pt, pph, r, T(0), pr, pth, o, hs, s, c);
  } else {
    rhs_schwarzschild<T, true>(mc, pt, pph, r, T(0), pr, pth, o, s, c);
    o.dt *= hs; o.dr *= hs; o.dth *= hs; o.dph *= hs; o.dpr *= hs; o.dpth *= hs;
  }
}

// Unscaled evaluation with sin and cos of theta supplied by the caller (Schwarzschild, Kerr): the stages of
// trace_rk4 obtain them from (sin, cos) theta_n by the addition theorems (sincos_add).
template <int METRIC, class T>
GP_HD void rhs_eval_sc(const MetricConst &mc, T pt, T pph, T r, T s, T c, T pr, T pth, RhsT<T> &o) {
  if (METRIC == METRIC_KERR) rhs_kerr<T, false, true>(mc, pt, pph, r, T(0), pr, pth, o, T(1), s, c);
  else rhs_schwarzschild<T, true>(mc, pt, pph, r, T(0), pr, pth, o, s, c);
}

// The mixed-precision form (cfg.precision = 2): the equations are evaluated in FP32 at the FP64 state
// rounded to FP32, the six derivatives come back in FP64 multiplied by hs.
template <int METRIC>
GP_HD void rhs_eval_fp32_scaled(const MetricConst &mc, double pt, double pph, double r, double th, double pr,
                                double pth, double hs, RhsT<double> &o) {
  RhsT<float> f;
  f.pw = 0.0f;
  rhs_eval<METRIC, true, float>(mc, (float)pt, (float)pph, (float)r, (float)th, (float)pr, (float)pth, f);
  o.dt = hs * (double)f.dt; o.dr = hs * (double)f.dr; o.dth = hs * (double)f.dth;
  o.dph = hs * (double)f.dph; o.dpr = hs * (double)f.dpr; o.dpth = hs * (double)f.dpth;
  o.s = (double)f.s; o.c = (double)f.c; o.H2 = (double)f.H2; o.is = (double)f.is; o.pw = (double)f.pw;
}

// ---- covariant metric at a point (host: observer tetrad, row a3) ------------------------------
// out: g_tt, g_tphi, g_phiphi, g_rr, g_thth
GP_HD void metric_cov(int metric, const MetricConst &mc, double r, double th, double g[5]) {
  double s = sin(th), c = cos(th);
  if (metric == METRIC_SCHW) {
    double F = 1.0 - 2.0 * mc.M / r;
    g[0] = -F; g[1] = 0.0; g[2] = r * r * s * s; g[3] = 1.0 / F; g[4] = r * r;
  } else if (metric == METRIC_KERR) {
    double Sig = r * r + mc.a2 * c * c, Del = r * r - 2.0 * mc.M * r + mc.a2;
    g[0] = -(1.0 - 2.0 * mc.M * r / Sig);
    g[1] = -2.0 * mc.M * mc.a * r * s * s / Sig;
    g[2] = (r * r + mc.a2 + 2.0 * mc.M * mc.a2 * r * s * s / Sig) * s * s;
    g[3] = Sig / Del;
    g[4] = Sig;
  } else {
    double x = (r - mc.M) * mc.mn_inv_k;
    MNCore<double> m = mn_core<double>(mc, x, c);
    double Del = mc.mn_k * mc.mn_k * (x * x - 1.0);
    g[0] = -m.f;
    g[1] = m.f * m.omega;
    g[2] = -m.f * m.omega * m.omega + Del * s * s / m.f;
    g[3] = m.E / (m.f * Del);
    g[4] = m.E / m.f;
  }
}

// ---- the 15-number table of gp_eval_metric (row a4 alone) -------------------------------------
// out15 = (g^tt, g^tphi, g^phiphi, g^rr, g^thth), d/dr of the five, d/dtheta of the five.
GP_HD void metric_inv15(int metric, const MetricConst &mc, double r, double th, double o[15]) {
  double s, c;
  sincos(th, &s, &c);
  if (metric == METRIC_SCHW) {
    double ir = 1.0 / r, ir2 = ir * ir, F = 1.0 - 2.0 * mc.M * ir, iF = 1.0 / F;
    double is2 = 1.0 / (s * s), Fr = 2.0 * mc.M * ir2;
    for (int i = 0; i < 15; ++i) o[i] = 0.0;
    o[0] = -iF; o[2] = ir2 * is2; o[3] = F; o[4] = ir2;
    o[5] = Fr * iF * iF; o[7] = -2.0 * ir2 * ir * is2; o[8] = Fr; o[9] = -2.0 * ir2 * ir;
    o[12] = -2.0 * c * ir2 * is2 / s;
  } else if (metric == METRIC_KERR) {
    // u = 1/Sigma, v = 1/Delta and their derivatives, then products
    const double a = mc.a, a2 = mc.a2, M = mc.M;
    double rr = r * r + a2, Sig = r * r + a2 * c * c, Del = rr - 2.0 * M * r;
    double u = 1.0 / Sig, v = 1.0 / Del, is2 = 1.0 / (s * s);
    double u_r = -2.0 * r * u * u, u_t = 2.0 * a2 * s * c * u * u, v_r = -2.0 * (r - M) * v * v;
    double T = rr * rr * v - a2 * s * s;                   // g^tt = -T u
    double T_r = 4.0 * r * rr * v + rr * rr * v_r, T_t = -2.0 * a2 * s * c;
    o[0] = -T * u; o[5] = -(T_r * u + T * u_r); o[10] = -(T_t * u + T * u_t);
    double X = -2.0 * M * a * r * v;                       // g^tphi = X u
    double X_r = -2.0 * M * a * (v + r * v_r);
    o[1] = X * u; o[6] = X_r * u + X * u_r; o[11] = X * u_t;
    double Y = is2 - a2 * v;                               // g^phiphi = Y u
    double Y_r = -a2 * v_r, Y_t = -2.0 * c * is2 / s;
    o[2] = Y * u; o[7] = Y_r * u + Y * u_r; o[12] = Y_t * u + Y * u_t;
    o[3] = Del * u; o[8] = 2.0 * (r - M) * u + Del * u_r; o[13] = Del * u_t;
    o[4] = u; o[9] = u_r; o[14] = u_t;
  } else {
    const double k = mc.mn_k;
    Dual2 x((r - mc.M) * mc.mn_inv_k, 1.0, 0.0), y(c, 0.0, 1.0);
    MNCore<Dual2> m = mn_core<Dual2>(mc, x, y);
    Dual2 Del = (k * k) * (sqr(x) - 1.0);
    Dual2 s2(s * s, 0.0, -2.0 * c);
    Dual2 fDs = m.f * recip(Del * s2);
    Dual2 fE = m.f * recip(m.E);
    Dual2 g[5];
    g[0] = fDs * sqr(m.omega) - recip(m.f);
    g[1] = fDs * m.omega;
    g[2] = fDs;
    g[3] = fE * Del;
    g[4] = fE;
    for (int i = 0; i < 5; ++i) {
      o[i] = g[i].v;
      o[5 + i] = g[i].dx * mc.mn_inv_k;
      o[10 + i] = -s * g[i].dy;
    }
  }
}

}  // namespace gp
#endif
