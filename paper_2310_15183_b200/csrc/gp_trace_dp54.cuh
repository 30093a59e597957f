// gp_trace_dp54.cuh — persistent Dormand-Prince 5(4) kernel (scheme 2; reading R10).
// Included by gp_trace.cuh.
//
// Loop shape (software-pipelined around the FSAL evaluation): every trip of the loop is
//   A  one evaluation of Hamilton's equations at each lane's PENDING state — the trial end
//      state of the attempt in flight, or the initial state of a freshly fetched ray;
//   B  the per-lane decision that needed it: error norm, accept / reject, step-size control,
//      termination, equator crossing, landing bookkeeping, record store, stop tests, monitors;
//   C  stages 2..6 of the next attempt (ordinary or landing) and its trial end state.
// A fresh ray therefore costs no evaluation outside the common stream, and a lane whose ray
// ended is refilled at the top of the next trip.
#ifndef GP_TRACE_DP54_CUH_
#define GP_TRACE_DP54_CUH_

namespace gp {
#if defined(__CUDACC__)

// Shared-memory parking lot for the state a ray resumes from after an equator landing step:
// trial state (r, th, pr, pth, t, ph, lambda), next step, raw k7 (6) and its monitor triple.
constexpr int kParkSlotsDp54 = 17;

template <int METRIC, bool DISK>
__global__ void __launch_bounds__(kBlock) trace_dp54(const __grid_constant__ TraceParams P) {
  extern __shared__ double park[];  // [kParkSlotsDp54][kBlock] when DISK
  const MetricConst &mc = P.mc;
  const int tid = threadIdx.x;

  // ---- per-lane ray state (registers) ----
  int mode = MODE_IDLE;
  long long slot = -1;
  double pt = 0.0, pph = 0.0;                         // constants of the ray
  double t = 0.0, r = 0.0, th = 0.0, ph = 0.0, pr = 0.0, pth = 0.0, lam = 0.0;  // y_n
  double k1t = 0.0, k1r = 0.0, k1th = 0.0, k1ph = 0.0, k1pr = 0.0, k1pth = 0.0;  // raw F(y_n)
  double h = 0.0;                                     // step of the attempt in flight / next attempt
  double target = 0.0;                                // landing target
  // pending (trial) state and the error sums that still lack the e7 k7 term
  double nt = 0.0, nr = 0.0, nth = 0.0, nph = 0.0, npr = 0.0, npth = 0.0, nlam = 0.0;
  double et = 0.0, er = 0.0, eth = 0.0, eph = 0.0, epr = 0.0, epth = 0.0;
  Monitors mo = {0.0, 0.0, 0.0, 1.0, 0.0, 0.0};
  unsigned n_acc = 0, n_rej = 0, n_cross = 0, n_rec = 0, n_land = 0, status = 0;
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
          // a2 + a3
          double alpha, beta;
          alpha_beta(P.cc, P.cc.ray_begin + slot * P.cc.ray_stride, alpha, beta);
          initial_momentum(P.cc, alpha, beta, pt, npr, npth, pph);
          nt = 0.0; nr = P.cc.r_obs; nth = P.cc.theta_obs; nph = P.cc.phi_obs; nlam = 0.0;
          mode = MODE_FRESH;
          n_acc = n_rej = n_cross = n_rec = n_land = 0;
          mo.h_max = 0.0; mo.q_drift = 0.0; mo.Q0 = 0.0;
          mo.sin_min = __longlong_as_double(0x7ff0000000000000LL);
          mo.err_margin = __longlong_as_double(0x7ff0000000000000LL);
        }
      }
    }
    if (!__any_sync(kFull, mode != MODE_IDLE)) break;

    if (mode != MODE_IDLE) {
      // ---- A: F at the pending state (stage 7 of the attempt in flight / k1 of a fresh ray) ----
      Rhs o7;
      rhs_eval<METRIC>(mc, pt, pph, nr, nth, npr, npth, o7);

      // ---- B: decisions ----
      bool finished = false;
      bool moved = false;   // y_n changed: run the stop tests' monitor on the new state
      double monH = 0.0, monQ = 0.0, monS = 0.0;
      if (mode == MODE_FRESH) {
        t = nt; r = nr; th = nth; ph = nph; pr = npr; pth = npth; lam = nlam;
        k1t = o7.dt; k1r = o7.dr; k1th = o7.dth; k1ph = o7.dph; k1pr = o7.dpr; k1pth = o7.dpth;
        h = P.h_cap_rel * P.cc.r_obs;       // R10 item 4
        monH = fabs(0.5 * o7.H2); monQ = carter_q<METRIC>(mc, pt, pph, npth, o7); monS = fabs(o7.s);
        mode = MODE_NORMAL;
        moved = true;
      } else if (mode == MODE_NORMAL) {
        // R10 items 1-3: scaled max-norm over the six evolving components,
        //   err = max_j |h (e_j + E7 k7_j)| / (atol + rtol max(|y_j|, |y+_j|)).
        // The largest ratio is found by cross-multiplication (num_j den_best > num_best den_j) and
        // divided once; a tie within rounding picks either of two equal ratios.
        double nm = fabs(h * (et + dp.E7 * o7.dt)), dn = fma(P.rtol, dmax(fabs(t), fabs(nt)), P.atol);
        double nsum = nm;
#define GP_ERR_TERM(e_, k7_, y_, ny_)                                            \
  {                                                                              \
    double n_ = fabs(h * ((e_) + dp.E7 * (k7_)));                                \
    double d_ = fma(P.rtol, dmax(fabs(y_), fabs(ny_)), P.atol);                  \
    nsum += n_;                                                                  \
    bool gt_ = n_ * dn > nm * d_;                                                \
    nm = gt_ ? n_ : nm;                                                          \
    dn = gt_ ? d_ : dn;                                                          \
  }
        GP_ERR_TERM(er, o7.dr, r, nr)
        GP_ERR_TERM(eth, o7.dth, th, nth)
        GP_ERR_TERM(eph, o7.dph, ph, nph)
        GP_ERR_TERM(epr, o7.dpr, pr, npr)
        GP_ERR_TERM(epth, o7.dpth, pth, npth)
#undef GP_ERR_TERM
        // finite test on the sums: any inf/NaN term makes them non-finite (numerators are >= 0)
        double ysum = ((nt + nr) + (nth + nph)) + (npr + npth);
        double err = div_nr(nm, dn, rcp_nr(dn));
        if (!finite_d(nsum) || !finite_d(ysum) || !finite_d(err)) {
          ++n_rej;
          h *= dp.fac_min;
        } else {
          mo.err_margin = dmin(mo.err_margin, fabs(err - 1.0));
          // fac = 0.9 err^(-1/5), clamped to [0.2, 5] (err = 0 gives 5); the clamp of err keeps the
          // FP32 seed of pow_m1_5 in range and changes nothing: 0.9 (1e-5)^-0.2 = 9 > 5, 0.9 (1e4)^-0.2 = 0.14 < 0.2
          double fac = dp.safety * pow_m1_5(dmin(dmax(dp.err_lo, err), dp.err_hi));
          fac = dmin(dmax(dp.fac_min, fac), dp.fac_max);
          if (err > 1.0) {
            ++n_rej;
            h *= fac;
          } else {
            ++n_acc;
            double hnext = dmin(h * fac, P.h_cap_rel * nr);
            if (nr > P.r_esc || nr < P.r_cap) {
              // O8: discard the step, land on the surface from y_n
              status = (nr > P.r_esc) ? GP_RAY_ESCAPED : GP_RAY_CAPTURED;
              target = (nr > P.r_esc) ? P.r_esc : P.r_cap;
              mode = MODE_LAND_R;
            } else {
              bool commit = true;
              if ((th - kHalfPi) * (nth - kHalfPi) < 0.0) {
                ++n_cross;
                if (DISK && n_rec < (unsigned)P.max_crossings) {
                  // O7: locate the crossing from y_n; resume from the parked trial state afterwards
                  double *pk = park + tid;
                  pk[0 * kBlock] = nr; pk[1 * kBlock] = nth; pk[2 * kBlock] = npr; pk[3 * kBlock] = npth;
                  pk[4 * kBlock] = nt; pk[5 * kBlock] = nph; pk[6 * kBlock] = lam + h; pk[7 * kBlock] = hnext;
                  pk[8 * kBlock] = o7.dt; pk[9 * kBlock] = o7.dr; pk[10 * kBlock] = o7.dth;
                  pk[11 * kBlock] = o7.dph; pk[12 * kBlock] = o7.dpr; pk[13 * kBlock] = o7.dpth;
                  pk[14 * kBlock] = fabs(0.5 * o7.H2);
                  pk[15 * kBlock] = carter_q<METRIC>(mc, pt, pph, npth, o7);
                  pk[16 * kBlock] = fabs(o7.s);
                  target = kHalfPi;
                  mode = MODE_LAND_TH;
                  commit = false;
                }
              }
              if (commit) {
                monH = fabs(0.5 * o7.H2); monQ = carter_q<METRIC>(mc, pt, pph, npth, o7); monS = fabs(o7.s);
                t = nt; r = nr; th = nth; ph = nph; pr = npr; pth = npth; lam += h;
                k1t = o7.dt; k1r = o7.dr; k1th = o7.dth; k1ph = o7.dph; k1pr = o7.dpr; k1pth = o7.dpth;
                h = hnext;
                moved = true;
              }
            }
          }
        }
      } else if (mode == MODE_LAND_R) {
        // landed on the exit surface: the record is the landed state (R14)
        t = nt; r = target; th = nth; ph = nph; pr = npr; pth = npth; lam = nlam;
        ++n_land;
        finished = true;
      } else {  // MODE_LAND_TH
        ++n_land;
        if (DISK) {
          double rc = nr;
          if (rc >= P.disk_r_in && rc <= P.disk_r_out) {
            P.disk[slot].r_cross[n_rec] = rc;
            P.disk[slot].g[n_rec] = kepler_g(mc, rc, pt, pph);
            ++n_rec;
          }
          const double *pk = park + tid;
          r = pk[0 * kBlock]; th = pk[1 * kBlock]; pr = pk[2 * kBlock]; pth = pk[3 * kBlock];
          t = pk[4 * kBlock]; ph = pk[5 * kBlock]; lam = pk[6 * kBlock]; h = pk[7 * kBlock];
          k1t = pk[8 * kBlock]; k1r = pk[9 * kBlock]; k1th = pk[10 * kBlock];
          k1ph = pk[11 * kBlock]; k1pr = pk[12 * kBlock]; k1pth = pk[13 * kBlock];
          monH = pk[14 * kBlock]; monQ = pk[15 * kBlock]; monS = pk[16 * kBlock];
        }
        mode = MODE_NORMAL;
        moved = true;
      }

      // stop tests in the oracle's order (R18, R10 item 5), then the monitors of the new state (R22)
      if (mode == MODE_NORMAL) {
        if ((long long)n_acc + (long long)n_rej >= P.max_steps ||
            (P.lambda_max > 0.0 && lam >= P.lambda_max)) {
          status = GP_RAY_MAXSTEPS;
          finished = true;
        } else if (h < dp.h_floor * dmax(1.0, fabs(lam))) {
          status = GP_RAY_STEP_UNDERFLOW;
          finished = true;
        } else if (moved) {
          monitor_apply<METRIC>(mo, monH, monQ, monS, n_acc == 0 && n_rej == 0);
        }
      }

      if (finished) {
        unsigned attempts = n_acc + n_rej;
        unsigned n_rhs = 1u + 6u * attempts + 5u * n_land;
        store_record(P.rays + slot, t, r, th, ph, pr, pth, lam, pt, pph, mo, status, n_acc, n_rej, n_cross,
                     n_rec, n_rhs);
        if (DISK) {
          const double qnan = __longlong_as_double(0x7ff8000000000000LL);
          for (unsigned i = n_rec; i < 3u; ++i) {
            P.disk[slot].r_cross[i] = qnan;
            P.disk[slot].g[i] = qnan;
          }
        }
        tot_rays += 1; tot_steps += attempts; tot_rhs += n_rhs;
        mode = MODE_IDLE;
      } else {
        // ---- C: stages 2..6 of the next attempt from (y_n, k1) ----
        // step and reciprocal selector: ordinary step s = h, divisor 1; landing s = target - y_w,
        // divisor F_w (w = r or theta)
        const bool land_r = (mode == MODE_LAND_R), land_th = (mode == MODE_LAND_TH);
        const bool landing = land_r || land_th;
        const double s = land_r ? (target - r) : (land_th ? (target - th) : h);
#define GP_INV(o_dr, o_dth) (landing ? 1.0 / (land_r ? (o_dr) : (o_dth)) : 1.0)
        double iv = GP_INV(k1r, k1th);
        const double K1r = k1r * iv, K1th = k1th * iv, K1pr = k1pr * iv, K1pth = k1pth * iv;
        double bt = dp.B1 * (k1t * iv), bph = dp.B1 * (k1ph * iv), bl = dp.B1 * iv;   // quadratures t, phi, lambda
        double qet = dp.E1 * (k1t * iv), qeph = dp.E1 * (k1ph * iv);
        Rhs o;
        // stage 2
        rhs_eval<METRIC>(mc, pt, pph, r + s * (dp.A21 * K1r), th + s * (dp.A21 * K1th),
                         pr + s * (dp.A21 * K1pr), pth + s * (dp.A21 * K1pth), o);
        iv = GP_INV(o.dr, o.dth);
        const double K2r = o.dr * iv, K2th = o.dth * iv, K2pr = o.dpr * iv, K2pth = o.dpth * iv;
        // stage 3
        rhs_eval<METRIC>(mc, pt, pph, r + s * (dp.A31 * K1r + dp.A32 * K2r),
                         th + s * (dp.A31 * K1th + dp.A32 * K2th),
                         pr + s * (dp.A31 * K1pr + dp.A32 * K2pr),
                         pth + s * (dp.A31 * K1pth + dp.A32 * K2pth), o);
        iv = GP_INV(o.dr, o.dth);
        const double K3r = o.dr * iv, K3th = o.dth * iv, K3pr = o.dpr * iv, K3pth = o.dpth * iv;
        bt += dp.B3 * (o.dt * iv); bph += dp.B3 * (o.dph * iv); bl += dp.B3 * iv;
        qet += dp.E3 * (o.dt * iv); qeph += dp.E3 * (o.dph * iv);
        // stage 4
        rhs_eval<METRIC>(mc, pt, pph, r + s * (dp.A41 * K1r + dp.A42 * K2r + dp.A43 * K3r),
                         th + s * (dp.A41 * K1th + dp.A42 * K2th + dp.A43 * K3th),
                         pr + s * (dp.A41 * K1pr + dp.A42 * K2pr + dp.A43 * K3pr),
                         pth + s * (dp.A41 * K1pth + dp.A42 * K2pth + dp.A43 * K3pth), o);
        iv = GP_INV(o.dr, o.dth);
        const double K4r = o.dr * iv, K4th = o.dth * iv, K4pr = o.dpr * iv, K4pth = o.dpth * iv;
        bt += dp.B4 * (o.dt * iv); bph += dp.B4 * (o.dph * iv); bl += dp.B4 * iv;
        qet += dp.E4 * (o.dt * iv); qeph += dp.E4 * (o.dph * iv);
        // stage 5
        rhs_eval<METRIC>(mc, pt, pph,
                         r + s * (dp.A51 * K1r + dp.A52 * K2r + dp.A53 * K3r + dp.A54 * K4r),
                         th + s * (dp.A51 * K1th + dp.A52 * K2th + dp.A53 * K3th + dp.A54 * K4th),
                         pr + s * (dp.A51 * K1pr + dp.A52 * K2pr + dp.A53 * K3pr + dp.A54 * K4pr),
                         pth + s * (dp.A51 * K1pth + dp.A52 * K2pth + dp.A53 * K3pth + dp.A54 * K4pth), o);
        iv = GP_INV(o.dr, o.dth);
        const double K5r = o.dr * iv, K5th = o.dth * iv, K5pr = o.dpr * iv, K5pth = o.dpth * iv;
        bt += dp.B5 * (o.dt * iv); bph += dp.B5 * (o.dph * iv); bl += dp.B5 * iv;
        qet += dp.E5 * (o.dt * iv); qeph += dp.E5 * (o.dph * iv);
        // stage 6
        rhs_eval<METRIC>(
            mc, pt, pph,
            r + s * (dp.A61 * K1r + dp.A62 * K2r + dp.A63 * K3r + dp.A64 * K4r + dp.A65 * K5r),
            th + s * (dp.A61 * K1th + dp.A62 * K2th + dp.A63 * K3th + dp.A64 * K4th + dp.A65 * K5th),
            pr + s * (dp.A61 * K1pr + dp.A62 * K2pr + dp.A63 * K3pr + dp.A64 * K4pr + dp.A65 * K5pr),
            pth + s * (dp.A61 * K1pth + dp.A62 * K2pth + dp.A63 * K3pth + dp.A64 * K4pth + dp.A65 * K5pth),
            o);
        iv = GP_INV(o.dr, o.dth);
        const double K6r = o.dr * iv, K6th = o.dth * iv, K6pr = o.dpr * iv, K6pth = o.dpth * iv;
        bt += dp.B6 * (o.dt * iv); bph += dp.B6 * (o.dph * iv); bl += dp.B6 * iv;
        qet += dp.E6 * (o.dt * iv); qeph += dp.E6 * (o.dph * iv);
#undef GP_INV
        // trial end state (5th-order solution; a7 = b) and the error sums without e7 k7
        nr = r + s * (dp.B1 * K1r + dp.B3 * K3r + dp.B4 * K4r + dp.B5 * K5r + dp.B6 * K6r);
        nth = th + s * (dp.B1 * K1th + dp.B3 * K3th + dp.B4 * K4th + dp.B5 * K5th + dp.B6 * K6th);
        npr = pr + s * (dp.B1 * K1pr + dp.B3 * K3pr + dp.B4 * K4pr + dp.B5 * K5pr + dp.B6 * K6pr);
        npth = pth + s * (dp.B1 * K1pth + dp.B3 * K3pth + dp.B4 * K4pth + dp.B5 * K5pth + dp.B6 * K6pth);
        nt = t + s * bt;
        nph = ph + s * bph;
        nlam = lam + s * bl;
        er = dp.E1 * K1r + dp.E3 * K3r + dp.E4 * K4r + dp.E5 * K5r + dp.E6 * K6r;
        eth = dp.E1 * K1th + dp.E3 * K3th + dp.E4 * K4th + dp.E5 * K5th + dp.E6 * K6th;
        epr = dp.E1 * K1pr + dp.E3 * K3pr + dp.E4 * K4pr + dp.E5 * K5pr + dp.E6 * K6pr;
        epth = dp.E1 * K1pth + dp.E3 * K3pth + dp.E4 * K4pth + dp.E5 * K5pth + dp.E6 * K6pth;
        et = qet;
        eph = qeph;
      }
    }
  }

  // totals (gp.h: counters[1] rays finished, [2] attempted steps, [3] RHS evaluations)
  if (tot_rays) {
    atomicAdd(P.counters + 1, tot_rays);
    atomicAdd(P.counters + 2, tot_steps);
    atomicAdd(P.counters + 3, tot_rhs);
  }
}

#endif  // __CUDACC__
}  // namespace gp
#endif
