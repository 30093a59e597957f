// gp_trace.cuh — the fused integrator kernels.
//
// One lane integrates one ray at a time and holds its whole state in registers; lanes pull
// ray slots from a global atomic counter (warp-aggregated) so that a lane whose ray ended
// refills at once and warps stay full in spite of divergent ray lengths (edge
// rays leave in < 1000 steps, others run 5e4..1e6).  Ordinary steps, landing steps onto the
// exit surface and landing steps onto the equator are ONE instruction stream: a landing step
// is a step of the same Runge-Kutta formula on dy/ds = F(y)/F_w(y) (Henon's device, DESIGN.md
// reading R14), so a per-lane reciprocal selector is all that differs.
//
//   classical RK4            PAPER.md L257-278 (eq 42-49), reading R9      -> trace_rk4
//   Dormand-Prince 5(4)      BASELINE.json configs[1-3], reading R10        -> trace_dp54
#ifndef GP_TRACE_CUH_
#define GP_TRACE_CUH_

#include "../../include/gp.h"
#include "gp_camera.cuh"
#include "gp_metric.cuh"

namespace gp {

struct TraceParams {
  MetricConst mc;
  CameraConst cc;
  int scheme;                       // 0 RK4 fixed h, 1 RK4 h = h_rel r, 2 DP5(4)
  int precision;                    // 0 FP64, 1 FP32 (RK4 schemes only)
  int max_crossings;                // 0 = disk off
  double h, h_rel, rtol, atol, h_cap_rel;
  long long max_steps;
  double lambda_max;   // +inf when the configuration has no affine budget (cfg.lambda_max <= 0)
  float h_f, h_rel_f;  // h and h_rel rounded to FP32, lambda_max rounded UP to FP32 (for any float x:
  float lambda_max_f;  // x >= lambda_max_f <=> (double)x >= lambda_max): the FP32 kernels' operands
  float pad_f_;
  double r_cap, r_esc;              // r_H (1 + eps_capture), r_escape
  double disk_r_in, disk_r_out;
  double ring_d;                    // half opening angle of the solid ring (> 0: object kind 2)
  gp_ray_record *rays;
  gp_disk_record *disk;
  unsigned long long *counters;
  // Segmented tracing of long rays (Manko-Novikov, scheme 2): after seg_steps attempted
  // steps a ray's state is parked in its own record and its slot appended to list_out; the next launch
  // (round + 1) takes its work from that list.  seg_steps = 0: off.
  long long seg_steps;
  int round;
  const long long *list_in;
  const unsigned long long *list_in_count;
  long long *list_out;
  unsigned long long *list_out_count;
};

enum { MODE_IDLE = 0, MODE_FRESH = 1, MODE_NORMAL = 2, MODE_LAND_R = 3, MODE_LAND_TH = 4, MODE_RESUME = 5 };
constexpr unsigned kRayParked = 255u;   // internal status of a record that holds a parked state (never left behind)

#if defined(__CUDACC__)
// Rows a2 + a3 for one ray: image-plane point, then the initial state of the selected camera.
// projection 0: the pinhole of gp_camera.cuh (every ray starts at the observer).
// projection 1: the paper's Euclidean screen: start point and direction on a
// flat screen in the xyz of eq 51-53, to Boyer-Lindquist by inverting eq 51-53 and differentiating
// the inverse, dt/dlambda from eq 54 (the root < 0), scaled to dt/dlambda = -1, lowered by eq 55.
// Kept out of line: it runs once per ray and must not weigh on the register allocation of the step loop.
__device__ __noinline__ void ray_birth_screen(const CameraConst &cc, const MetricConst &mc, double alpha,
                                              double beta, double *out7) {
  const double a = cc.a_cam;
  double X[3], V[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double off = alpha * cc.eph[i] + beta * cc.eup[i];
    X[i] = cc.r_obs * cc.chat[i] + off;
    V[i] = cc.k2 * off - cc.chat[i];
  }
  const double w = X[0] * X[0] + X[1] * X[1] + X[2] * X[2] - a * a;
  const double r = sqrt(0.5 * (w + sqrt(w * w + 4.0 * a * a * X[2] * X[2])));
  const double th = acos(X[2] / r);
  const double ph = atan2(X[1], X[0]);
  double sth, cth, sph, cph;
  sincos(th, &sth, &cth);
  sincos(ph, &sph, &cph);
  const double R = sqrt(r * r + a * a), Sig = r * r + a * a * cth * cth;
  const double u = V[0] * cph + V[1] * sph;
  double dph = (V[1] * cph - V[0] * sph) / (R * sth);
  double dr = R * (r * sth * u + R * cth * V[2]) / Sig;
  double dth = (R * cth * u - r * sth * V[2]) / Sig;
  double g[5];
  metric_cov(cc.metric_id, mc, r, th, g);
  const double S = g[3] * dr * dr + g[4] * dth * dth + g[2] * dph * dph;
  const double B = g[1] * dph;
  const double dt = (sqrt(B * B - g[0] * S) - B) / g[0];
  const double sc = -1.0 / dt;
  dr *= sc; dth *= sc; dph *= sc;
  out7[0] = r; out7[1] = th; out7[2] = ph;
  out7[3] = g[1] * dph - g[0];
  out7[4] = g[3] * dr;
  out7[5] = g[4] * dth;
  out7[6] = g[2] * dph - g[1];
}

__device__ __forceinline__ void ray_birth(const CameraConst &cc, const MetricConst &mc, long long ray, double &r,
                                          double &th, double &ph, double &pt, double &pr, double &pth,
                                          double &pph) {
  double alpha, beta;
  alpha_beta(cc, ray, alpha, beta);
  if (cc.projection == 0) {
    initial_momentum(cc, alpha, beta, pt, pr, pth, pph);
    r = cc.r_obs; th = cc.theta_obs; ph = cc.phi_obs;
  } else {
    double o[7];
    ray_birth_screen(cc, mc, alpha, beta, o);
    r = o[0]; th = o[1]; ph = o[2]; pt = o[3]; pr = o[4]; pth = o[5]; pph = o[6];
  }
}
#endif

#ifndef GP_BLOCK
#define GP_BLOCK 128
#endif
constexpr int kBlock = GP_BLOCK;
constexpr unsigned kFull = 0xffffffffu;
constexpr double kHalfPi = 1.57079632679489661923;

// Dormand & Prince (1980) 5(4) pair, reading R10.  The coefficients sit in __constant__ memory so
// that DFMA/DMUL take them as c[bank][offset] operands: as literals each use cost two UMOVs
// (profiles/r01: 17 % of all warp instructions).
// Rows start on 16-byte boundaries so that the compiler can fetch two coefficients per LDCU.128.
struct alignas(16) DpTableau {
  double A21, pad0_;
  double A31, A32;
  double A41, A42, A43, pad1_;
  double A51, A52, A53, A54;
  double A61, A62, A63, A64, A65, pad2_;
  double B1, B3, B4, B5, B6, pad3_;
  double E1, E3, E4, E5, E6, E7;
  double safety, fac_min, fac_max, err_lo, err_hi, h_floor;  // controller constants, R10 items 3 and 5
  double sixth;                                              // RK4 weight 1/6 (eq 44)
};

#if defined(__CUDACC__)
__constant__ DpTableau dp = {
    1.0 / 5.0, 0.0,
    3.0 / 40.0, 9.0 / 40.0,
    44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0.0,
    19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0,
    9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0.0,
    35.0 / 384.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0, 0.0,
    71.0 / 57600.0, -71.0 / 16695.0, 71.0 / 1920.0, -17253.0 / 339200.0, 22.0 / 525.0, -1.0 / 40.0,
    0.9, 0.2, 5.0, 1.0e-5, 1.0e4, 1.0e-14,
    1.0 / 6.0};
#endif

#if defined(__CUDACC__)

__device__ __forceinline__ bool finite_d(double x) { return fabs(x) <= 1.79769313486231570815e308; }

// 256-bit store of four doubles (one 32-byte sector per instruction; row a11).
__device__ __forceinline__ void store4(double *p, double a, double b, double c, double d) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// Warp-aggregated work fetch (row a1): one atomic per warp per refill round.  Returns the output
// slot for this lane or -1 when the image is exhausted.
__device__ __forceinline__ long long fetch_slot(unsigned need_mask, bool need, unsigned long long *counter,
                                                long long ray_count) {
  const unsigned lane = threadIdx.x & 31u;
  const int leader = __ffs(need_mask) - 1;
  unsigned long long base = 0;
  if ((int)lane == leader) base = atomicAdd(counter, (unsigned long long)__popc(need_mask));
  base = __shfl_sync(kFull, base, leader);
  if (!need) return -1;
  // Slots are handed out in increasing order.  Longest-rays-first orders were measured (centre-out:
  // 1.5 % slower on the Kerr headline, 0.8 % faster on Manko-Novikov config 4; middle rows first: no
  // change) and not kept: the 3.9 % tail of the 1024^2 headline is the granularity of 13.8 rays per
  // lane, not the order they come in.
  long long slot = (long long)(base + (unsigned long long)__popc(need_mask & ((1u << lane) - 1u)));
  return slot < ray_count ? slot : -1;
}

// Prograde Keplerian emitter on the equator (eq 56 in closed form; L372,
// eq 57; readings R19/R20): g = (p.u_obs)/(p.u_emit) = 1/[u^t (p_t + Omega_K p_phi)].
__device__ __forceinline__ double kepler_g_closed(const MetricConst &mc, double r, double pt, double pph) {
  double sM = sqrt(mc.M);
  double sr = sqrt(r);
  double r32 = r * sr;
  double den = r32 + mc.a * sM;
  double Om = sM / den;
  double ut = den / (sqrt(r32) * sqrt(r32 - 3.0 * mc.M * sr + 2.0 * mc.a * sM));
  return 1.0 / (ut * (pt + Om * pph));
}

// The same emitter from eq 56 itself, for metrics without a closed form (Manko-Novikov): with
// p_t = -1 the circular-orbit condition dp_r/dlambda = 0 is the quadratic
// d_r g^{phi phi} p_phi^2 - 2 d_r g^{t phi} p_phi + d_r g^{tt} = 0; the derivatives come from the dual
// numbers of metric_inv15; the root with Omega > 0 is taken and p normalised to p^2 = -1.  NaN when
// there is no circular orbit at r.  Runs once per recorded crossing: kept out of line.
__device__ __noinline__ double kepler_g_general(int metric, const MetricConst &mc, double r, double pt, double pph) {
  double g[15];
  metric_inv15(metric, mc, r, kHalfPi, g);
  const double gtt = g[0], gtp = g[1], gpp = g[2];
  const double A = g[7], B = g[6], C = g[5];
  const double disc = B * B - A * C;
  double Om_best = 0.0, ut_best = 0.0;
  bool found = false;
  if (disc >= 0.0) {
    const double sq = sqrt(disc);
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      double pe = (B + (k == 0 ? sq : -sq)) / A;
      double ut_raw = gtp * pe - gtt;
      double uph_raw = gpp * pe - gtp;
      double N = -(gtt - 2.0 * gtp * pe + gpp * pe * pe);
      double Om = uph_raw / ut_raw;
      if (N > 0.0 && ut_raw > 0.0 && Om > 0.0) {
        Om_best = Om;
        ut_best = ut_raw / sqrt(N);
        found = true;
      }
    }
  }
  if (!found) return __longlong_as_double(0x7ff8000000000000LL);
  return 1.0 / (ut_best * (pt + Om_best * pph));
}

template <int METRIC>
__device__ __forceinline__ double kepler_g(const MetricConst &mc, double r, double pt, double pph) {
  if (METRIC == METRIC_MN) return kepler_g_general(METRIC_MN, mc, r, pt, pph);
  return kepler_g_closed(mc, r, pt, pph);
}

// Progress stamps ("steady-state rate excluding the final tail"): counters[4] =
// %globaltimer (ns) when the kernel starts, [5] = when 99 % of the rays have finished, [7] = when
// the last block leaves; [6] counts finished rays live (one atomic per ray: ~5e7/s against a limit far
// above that).
__device__ __forceinline__ unsigned long long global_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
  return t;
}
__device__ __forceinline__ void stamp_start(unsigned long long *counters) {
  if (blockIdx.x == 0 && threadIdx.x == 0 && counters[4] == 0ull) counters[4] = global_ns();   // first round only
}
__device__ __forceinline__ void stamp_ray_done(unsigned long long *counters, long long ray_count) {
  const unsigned long long done = atomicAdd(counters + 6, 1ull) + 1ull;
  if ((long long)done == ray_count - ray_count / 100) counters[5] = global_ns();
}
__device__ __forceinline__ void stamp_end(unsigned long long *counters) {
  if (threadIdx.x == 0) atomicMax(counters + 7, global_ns());
}

// Monitors of row a10 carried per lane.
template <class T>
struct MonitorsT {
  T h_max, q_drift, Q0, iQ0, sin_min, err_margin;
};
typedef MonitorsT<double> Monitors;

__device__ __forceinline__ float dmax(float run, float cand) { return cand > run ? cand : run; }
__device__ __forceinline__ float dmin(float run, float cand) { return cand < run ? cand : run; }
__device__ __forceinline__ bool finite_d(float x) { return fabsf(x) <= 3.402823466e38f; }

// Carter constant, exact off shell (reading R23): Q = p_th^2 + c^2 (p_ph^2/s^2 - a^2 p_t^2) - 2 a^2 c^2 H.
template <int METRIC, class T>
__device__ __forceinline__ T carter_q(const MetricConst &mc, T pt, T pph, T pth, const RhsT<T> &o) {
  if (METRIC == METRIC_MN) return T(0);
  if (METRIC == METRIC_KERR) {
    // c^2 (p_ph^2/s^2 - a^2 p_t^2) = W^2 - (p_ph + a p_t)^2 with W = p_ph/s + a s p_t, and p_th^2 + W^2 is
    // a by-product of rhs_kerr: five operations instead of eleven, every step
    T l = ffma((T)mc.a, pt, pph);
    return ffma(-((T)mc.a2 * o.c) * o.c, o.H2, o.pw - l * l);
  }
  T c2 = o.c * o.c;
  return pth * pth + c2 * (pph * pph * o.is * o.is);
}

template <int METRIC, class T>
__device__ __forceinline__ void monitor_apply(MonitorsT<T> &mo, T absH, T Q, T abss, bool first) {
  mo.h_max = dmax(mo.h_max, absH);
  mo.sin_min = dmin(mo.sin_min, abss);
  if (METRIC != METRIC_MN) {
    if (first) mo.Q0 = Q;
    if (first) mo.iQ0 = frcp(dmax(T(1), (T)fabs(Q)));
    T d = (T)fabs(Q - mo.Q0) * mo.iQ0;
    mo.q_drift = dmax(mo.q_drift, d);
  }
}

// Row a11: pack and store the 128-byte record with four 256-bit stores.
__device__ __forceinline__ void store_record(gp_ray_record *rec, double t, double r, double th, double ph,
                                             double pr, double pth, double lam, double pt, double pph,
                                             const Monitors &mo, unsigned status, unsigned n_acc,
                                             unsigned n_rej, unsigned n_cross, unsigned n_rec,
                                             unsigned n_rhs) {
  double *p = reinterpret_cast<double *>(rec);
  double w0 = __hiloint2double((int)n_acc, (int)status);      // little endian: status, n_accepted
  double w1 = __hiloint2double((int)n_cross, (int)n_rej);     // n_rejected, n_equator_crossings
  double w2 = __hiloint2double((int)n_rhs, (int)n_rec);       // n_disk_recorded, n_rhs
  store4(p, t, r, th, ph);
  store4(p + 4, lam, w0, pr, pth);
  store4(p + 8, pt, pph, mo.h_max, mo.q_drift);
  store4(p + 12, mo.sin_min, mo.err_margin, w1, w2);
}

#endif  // __CUDACC__
}  // namespace gp

#include "gp_trace_dp54.cuh"
#include "gp_trace_rk4.cuh"

#endif
