// gp_trace_rk4.cuh — persistent classical RK4 kernel (schemes 0 and 1; PAPER.md L257-278,
// eq 42-49 with reading R9; step h fixed, or h_n = h_rel r_n per reading R17).
// Included by gp_trace.cuh.
//
// Every trip of the loop is one RK4 step per lane: an ordinary step, or a landing step of the
// same formula on dy/ds = F/F_w (reading R14).  Reading R31: in an ordinary step each state the
// equations are evaluated at is first tested against the capture radius; the first hit ends the
// ray as CAPTURED (then one landing step from y_n).
#ifndef GP_TRACE_RK4_CUH_
#define GP_TRACE_RK4_CUH_

namespace gp {
#if defined(__CUDACC__)

constexpr int kParkSlotsRk4 = 7;  // trial state (r, th, pr, pth, t, ph, lambda) across an equator landing

template <int METRIC, bool DISK>
__global__ void __launch_bounds__(kBlock) trace_rk4(const __grid_constant__ TraceParams P) {
  extern __shared__ double park[];  // [kParkSlotsRk4][kBlock] when DISK
  const MetricConst &mc = P.mc;
  const int tid = threadIdx.x;

  int mode = MODE_IDLE;
  long long slot = -1;
  double pt = 0.0, pph = 0.0;
  double t = 0.0, r = 0.0, th = 0.0, ph = 0.0, pr = 0.0, pth = 0.0, lam = 0.0;
  double target = 0.0;
  Monitors mo = {0.0, 0.0, 0.0, 1.0, 0.0, 0.0};
  unsigned n_acc = 0, n_cross = 0, n_rec = 0, n_land = 0, status = 0;
  bool exhausted = false;
  unsigned long long tot_rays = 0, tot_steps = 0, tot_rhs = 0;

  for (;;) {
    // ---- a1: refill idle lanes ----
    const bool need = (mode == MODE_IDLE) && !exhausted;
    const unsigned need_mask = __ballot_sync(kFull, need);
    if (need_mask) {
      const long long got = fetch_slot(need_mask, need, P.counters, P.cc.ray_count);
      if (need) {
        slot = got;
        if (slot < 0) {
          exhausted = true;
        } else {
          double alpha, beta;
          alpha_beta(P.cc, P.cc.ray_begin + slot * P.cc.ray_stride, alpha, beta);
          initial_momentum(P.cc, alpha, beta, pt, pr, pth, pph);
          t = 0.0; r = P.cc.r_obs; th = P.cc.theta_obs; ph = P.cc.phi_obs; lam = 0.0;
          mode = MODE_NORMAL;
          n_acc = n_cross = n_rec = n_land = 0;
          mo.h_max = 0.0; mo.q_drift = 0.0; mo.Q0 = 0.0;
          mo.sin_min = __longlong_as_double(0x7ff0000000000000LL);
          mo.err_margin = __longlong_as_double(0x7ff0000000000000LL);
        }
      }
    }
    if (!__any_sync(kFull, mode != MODE_IDLE)) break;

    if (mode != MODE_IDLE) {
      bool finished = false;
      // stop tests at the top of every ordinary step (R18)
      if (mode == MODE_NORMAL &&
          ((long long)n_acc >= P.max_steps || (P.lambda_max > 0.0 && lam >= P.lambda_max))) {
        status = GP_RAY_MAXSTEPS;
        finished = true;
      }
      if (!finished) {
        const bool normal = (mode == MODE_NORMAL);
        const bool land_r = (mode == MODE_LAND_R);
        const double s = normal ? (P.scheme == 0 ? P.h : P.h_rel * r) : (land_r ? (target - r) : (target - th));
        // Landing steps are 1 in several hundred: their divisor work (Henon's 1/F_w) sits behind a
        // warp-uniform branch taken only when some lane of this convergence group is landing.
        const bool any_land = __any_sync(__activemask(), !normal);
        double sl = 1.0;  // weighted sum of 1/F_w: d(lambda)/ds of a landing step (unused otherwise)
#define GP_HENON(weight, first)                                                   \
  if (any_land) {                                                                 \
    double iv = normal ? 1.0 : rcp_nr(land_r ? o.dr : o.dth);                     \
    o.dt *= iv; o.dr *= iv; o.dth *= iv; o.dph *= iv; o.dpr *= iv; o.dpth *= iv;  \
    sl = (first) ? iv : sl + (weight) * iv;                                       \
  }
        Rhs o;
        // k1 = F(y_n)
        rhs_eval<METRIC>(mc, pt, pph, r, th, pr, pth, o);
        if (normal)
          monitor_apply<METRIC>(mo, fabs(0.5 * o.H2), carter_q<METRIC>(mc, pt, pph, pth, o), fabs(o.s),
                                n_acc == 0);
        GP_HENON(1.0, true)
        double st = o.dt, sr = o.dr, sth = o.dth, sph = o.dph, spr = o.dpr, spth = o.dpth;  // k1 + 2k2 + 2k3 + k4
        const double hs = 0.5 * s;
        // k2 = F(y_n + h/2 k1)
        double yr = r + hs * o.dr;
        bool captured = normal && (yr < P.r_cap);
        rhs_eval<METRIC>(mc, pt, pph, yr, th + hs * o.dth, pr + hs * o.dpr, pth + hs * o.dpth, o);
        GP_HENON(2.0, false)
        st += 2.0 * o.dt; sr += 2.0 * o.dr; sth += 2.0 * o.dth; sph += 2.0 * o.dph; spr += 2.0 * o.dpr;
        spth += 2.0 * o.dpth;
        // k3 = F(y_n + h/2 k2)
        yr = r + hs * o.dr;
        captured = captured || (normal && (yr < P.r_cap));
        rhs_eval<METRIC>(mc, pt, pph, yr, th + hs * o.dth, pr + hs * o.dpr, pth + hs * o.dpth, o);
        GP_HENON(2.0, false)
        st += 2.0 * o.dt; sr += 2.0 * o.dr; sth += 2.0 * o.dth; sph += 2.0 * o.dph; spr += 2.0 * o.dpr;
        spth += 2.0 * o.dpth;
        // k4 = F(y_n + h k3)
        yr = r + s * o.dr;
        captured = captured || (normal && (yr < P.r_cap));
        rhs_eval<METRIC>(mc, pt, pph, yr, th + s * o.dth, pr + s * o.dpr, pth + s * o.dpth, o);
        GP_HENON(1.0, false)
        st += o.dt; sr += o.dr; sth += o.dth; sph += o.dph; spr += o.dpr; spth += o.dpth;
#undef GP_HENON
        const double w = s * dp.sixth;
        const double nt = t + w * st, nr = r + w * sr, nth = th + w * sth, nph = ph + w * sph,
                     npr = pr + w * spr, npth = pth + w * spth;

        if (normal) {
          const double ysum = ((nt + nr) + (nth + nph)) + (npr + npth);
          const bool nonfinite = !captured && !finite_d(ysum);
          if (!nonfinite) ++n_acc;
          if (nonfinite) {
            status = GP_RAY_NONFINITE;   // record = last finite state y_n
            finished = true;
          } else if (captured || nr > P.r_esc || nr < P.r_cap) {
            const bool esc = !captured && nr > P.r_esc;
            status = esc ? GP_RAY_ESCAPED : GP_RAY_CAPTURED;
            target = esc ? P.r_esc : P.r_cap;
            mode = MODE_LAND_R;
          } else {
            bool commit = true;
            if ((th - kHalfPi) * (nth - kHalfPi) < 0.0) {
              ++n_cross;
              if (DISK && n_rec < (unsigned)P.max_crossings) {
                double *pk = park + tid;
                pk[0 * kBlock] = nr; pk[1 * kBlock] = nth; pk[2 * kBlock] = npr; pk[3 * kBlock] = npth;
                pk[4 * kBlock] = nt; pk[5 * kBlock] = nph; pk[6 * kBlock] = lam + s;
                target = kHalfPi;
                mode = MODE_LAND_TH;
                commit = false;
              }
            }
            if (commit) {
              t = nt; r = nr; th = nth; ph = nph; pr = npr; pth = npth; lam += s;
            }
          }
        } else if (land_r) {
          t = nt; r = target; th = nth; ph = nph; pr = npr; pth = npth; lam = lam + w * sl;
          ++n_land;
          finished = true;
        } else {  // MODE_LAND_TH
          ++n_land;
          if (DISK) {
            const double rc = nr;
            if (rc >= P.disk_r_in && rc <= P.disk_r_out) {
              P.disk[slot].r_cross[n_rec] = rc;
              P.disk[slot].g[n_rec] = kepler_g(mc, rc, pt, pph);
              ++n_rec;
            }
            const double *pk = park + tid;
            r = pk[0 * kBlock]; th = pk[1 * kBlock]; pr = pk[2 * kBlock]; pth = pk[3 * kBlock];
            t = pk[4 * kBlock]; ph = pk[5 * kBlock]; lam = pk[6 * kBlock];
          }
          mode = MODE_NORMAL;
        }
      }

      if (finished) {
        const unsigned n_rhs = 4u * n_acc + 3u * n_land;
        store_record(P.rays + slot, t, r, th, ph, pr, pth, lam, pt, pph, mo, status, n_acc, 0u, n_cross, n_rec,
                     n_rhs);
        if (DISK) {
          const double qnan = __longlong_as_double(0x7ff8000000000000LL);
          for (unsigned i = n_rec; i < 3u; ++i) {
            P.disk[slot].r_cross[i] = qnan;
            P.disk[slot].g[i] = qnan;
          }
        }
        tot_rays += 1; tot_steps += n_acc; tot_rhs += n_rhs;
        mode = MODE_IDLE;
      }
    }
  }

  if (tot_rays) {
    atomicAdd(P.counters + 1, tot_rays);
    atomicAdd(P.counters + 2, tot_steps);
    atomicAdd(P.counters + 3, tot_rhs);
  }
}

#endif  // __CUDACC__
}  // namespace gp
#endif
