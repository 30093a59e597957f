// gp_orbits.cuh — orbits from explicit initial states (section 3.2.1 and Fig 1:
// time-like test orbits, the same Hamilton's equations with H = -1/2; L719, Fig 11: neighbouring
// null orbits).  SURVEY.md section 8(f) NEXT-3; contract in include/gp.h (gp_integrate_orbits).
//
// One lane per orbit, Dormand-Prince 5(4) with the controller of reading R10, every attempted step
// min(h, h_max, lambda_next - lambda) so that the state is sampled exactly at
// lambda_k = (k+1) lambda_end / n_samples; a step cut short by a sample time keeps the controller's
// previous proposal when that is larger.  Not the hot path: orbits are few and equally long, so this
// is the plain register-resident form of the integrator (no work queue, no shared memory).
#ifndef GP_ORBITS_CUH_
#define GP_ORBITS_CUH_

#include "gp_trace.cuh"

namespace gp {
#if defined(__CUDACC__)

struct OrbitParams {
  MetricConst mc;
  double rtol, atol, h0, h_max, lambda_end, r_cap;
  long long n, n_samples, max_steps;
  const double *states8;
  double *samples;          // n * n_samples * 8: t, r, theta, phi, p_r, p_theta, 2H, lambda
  unsigned *status;         // n
  unsigned long long *n_steps;  // n
};

template <int METRIC>
__global__ void __launch_bounds__(128) k_integrate_orbits(const __grid_constant__ OrbitParams P) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P.n) return;
  const MetricConst &mc = P.mc;
  const double *st = P.states8 + 8 * i;
  double *out = P.samples + 8 * P.n_samples * i;
  const double qnan = __longlong_as_double(0x7ff8000000000000LL);
  for (long long j = 0; j < 8 * P.n_samples; ++j) out[j] = qnan;
  const double pt = st[4], pph = st[7];
  double y[6] = {st[0], st[1], st[2], st[3], st[5], st[6]};   // t, r, th, ph, pr, pth
  double k[7][6];
  Rhs o;
  auto F = [&](const double *yy, double *dy) {
    rhs_eval<METRIC, true>(mc, pt, pph, yy[1], yy[2], yy[4], yy[5], o);
    dy[0] = o.dt; dy[1] = o.dr; dy[2] = o.dth; dy[3] = o.dph; dy[4] = o.dpr; dy[5] = o.dpth;
  };
  F(y, k[0]);
  double lam = 0.0, h = P.h0;
  long long next = 0;
  unsigned long long steps = 0;
  unsigned stat = 0;
  const double A[7][6] = {{0, 0, 0, 0, 0, 0},
                          {dp.A21, 0, 0, 0, 0, 0},
                          {dp.A31, dp.A32, 0, 0, 0, 0},
                          {dp.A41, dp.A42, dp.A43, 0, 0, 0},
                          {dp.A51, dp.A52, dp.A53, dp.A54, 0, 0},
                          {dp.A61, dp.A62, dp.A63, dp.A64, dp.A65, 0},
                          {dp.B1, 0.0, dp.B3, dp.B4, dp.B5, dp.B6}};
  const double E[7] = {dp.E1, 0.0, dp.E3, dp.E4, dp.E5, dp.E6, dp.E7};
  while (next < P.n_samples) {
    if ((long long)steps >= P.max_steps) { stat = GP_RAY_MAXSTEPS; break; }
    if (h < dp.h_floor * dmax(1.0, fabs(lam))) { stat = GP_RAY_STEP_UNDERFLOW; break; }
    const double lam_next = (double)(next + 1) * P.lambda_end / (double)P.n_samples;
    const double room = lam_next - lam;
    double hs = dmin(h, P.h_max);
    const bool cut = !(hs < room);
    if (cut) hs = room;
    double ynew[6], tmp[6];
#pragma unroll
    for (int s = 1; s < 7; ++s) {
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        double acc = 0.0;
#pragma unroll
        for (int j = 0; j < s; ++j) acc = fma(A[s][j], k[j][c], acc);
        tmp[c] = fma(hs, acc, y[c]);
      }
      if (s == 6) {
#pragma unroll
        for (int c = 0; c < 6; ++c) ynew[c] = tmp[c];
      }
      F(tmp, k[s]);
    }
    ++steps;
    double err = 0.0, ysum = 0.0, esum = 0.0;
#pragma unroll
    for (int c = 0; c < 6; ++c) {
      double acc = 0.0;
#pragma unroll
      for (int j = 0; j < 7; ++j) acc = fma(E[j], k[j][c], acc);
      double e = fabs(hs * acc) / (P.atol + P.rtol * dmax(fabs(y[c]), fabs(ynew[c])));
      esum += e;
      ysum += ynew[c];
      err = dmax(err, e);
    }
    if (!finite_d(esum) || !finite_d(ysum)) { h = hs * dp.fac_min; continue; }
    double fac = dp.safety * pow_m1_5(dmin(dmax(dp.err_lo, err), dp.err_hi));
    fac = dmin(dmax(dp.fac_min, fac), dp.fac_max);
    if (err > 1.0) { h = hs * fac; continue; }
    const double hnew = hs * fac;
    h = cut ? dmax(h, hnew) : hnew;
#pragma unroll
    for (int c = 0; c < 6; ++c) { y[c] = ynew[c]; k[0][c] = k[6][c]; }
    lam = cut ? lam_next : lam + hs;
    if (y[1] < P.r_cap) { stat = GP_RAY_CAPTURED; break; }
    if (cut) {
      double *s8 = out + 8 * next;
      const double H2 = pt * k[0][0] + y[4] * k[0][1] + y[5] * k[0][2] + pph * k[0][3];
      store4(s8, y[0], y[1], y[2], y[3]);
      store4(s8 + 4, y[4], y[5], H2, lam);
      ++next;
    }
  }
  P.status[i] = stat;
  P.n_steps[i] = steps;
}

#endif  // __CUDACC__
}  // namespace gp
#endif
