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

// Shared-memory plan, per lane.  Registers hold only what every stage
// touches; the rest lives in shared memory so that five blocks (20 warps) fit per SM:
//   K area   8 x double2   stage slopes K2..K5 of (r, th) and (p_r, p_th); K1 and the newest K stay
//                          in registers.  128-bit accesses, [slot][lane] layout: conflict-free.
//   cold     kColdSlots x double   state the stages never read: t, phi, lambda, the monitors, the
//                          landing target, k1 of the two quadratures, the per-lane totals.
//   park     17 x double   (DISK only) what a ray resumes from after an equator landing step:
//                          trial state (r, th, pr, pth, t, ph, lambda), next step, raw k7 (6) and
//                          its monitor triple.
enum { C_T = 0, C_PH, C_LAM, C_HMAX, C_QDRIFT, C_Q0, C_IQ0, C_SINMIN, C_MARGIN, C_TARGET, C_K1T, C_K1PH,
       C_TOT_RAYS, C_TOT_STEPS, C_TOT_RHS, kColdSlots };
constexpr int kKSlots2 = 8;
constexpr int kParkSlotsDp54 = 17;
constexpr size_t dp54_smem_bytes(bool disk) {
  return sizeof(double) * kBlock * (2 * kKSlots2 + kColdSlots + (disk ? kParkSlotsDp54 : 0));
}
// Resident blocks per SM the register allocation is held to (4 -> <= 128 registers, no spills for
// Schwarzschild and Kerr; the Manko-Novikov duals need 2 -> <= 255).  Measured on B200 (headline):
// 3 blocks 48.7, 4 blocks 51.6, 5 blocks (70 B of spills) 49.6 M geodesics/s.
#ifndef GP_DP54_MIN_BLOCKS
#define GP_DP54_MIN_BLOCKS 4
#endif
#ifndef GP_DP54_MIN_BLOCKS_MN
#define GP_DP54_MIN_BLOCKS_MN 2
#endif

// Shared-memory accessors by 32-bit shared-window address.  asm volatile keeps every access (the
// compiler would otherwise forward the stored K's back into registers and spill) and their order.
__device__ __forceinline__ void sts1(unsigned a, double x) {
  asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(x));
}
__device__ __forceinline__ double lds1(unsigned a) {
  double x;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(x) : "r"(a));
  return x;
}
__device__ __forceinline__ void sts2(unsigned a, double x, double y) {
  asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(x), "d"(y));
}
__device__ __forceinline__ void lds2(unsigned a, double &x, double &y) {
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(x), "=d"(y) : "r"(a));
}

template <int METRIC, bool DISK>
__global__ void __launch_bounds__(kBlock, METRIC == METRIC_MN ? GP_DP54_MIN_BLOCKS_MN : GP_DP54_MIN_BLOCKS)
trace_dp54(const __grid_constant__ TraceParams P) {
  extern __shared__ double2 smem2[];
  const MetricConst &mc = P.mc;
  const int tid = threadIdx.x;
  const unsigned sm_k = (unsigned)__cvta_generic_to_shared(smem2) + 16u * tid;                  // + 16 kBlock slot
  const unsigned sm_c = (unsigned)__cvta_generic_to_shared(smem2 + kKSlots2 * kBlock) + 8u * tid;  // + 8 kBlock slot
  const unsigned sm_p = sm_c + 8u * kBlock * kColdSlots;
#define KS(slot) (sm_k + 16u * kBlock * (slot))
#define CS(slot) (sm_c + 8u * kBlock * (slot))
#define PS(slot) (sm_p + 8u * kBlock * (slot))

  // ---- per-lane ray state (registers) ----
  int mode = MODE_IDLE;
  long long slot = -1;
  double pt = 0.0, pph = 0.0;                         // constants of the ray
  double r = 0.0, th = 0.0, pr = 0.0, pth = 0.0;      // y_n, the part Hamilton's equations read
  double k1r = 0.0, k1th = 0.0, k1pr = 0.0, k1pth = 0.0;  // raw F(y_n), same part
  double h = 0.0;                                     // step of the attempt in flight / next attempt
  // pending (trial) state and the error sums that still lack the e7 k7 term
  double nt = 0.0, nr = 0.0, nth = 0.0, nph = 0.0, npr = 0.0, npth = 0.0, nlam = 0.0;
  double et = 0.0, er = 0.0, eth = 0.0, eph = 0.0, epr = 0.0, epth = 0.0;
  unsigned n_acc = 0, n_rej = 0, n_cross = 0, n_rec = 0, n_land = 0, status = 0;
  bool exhausted = false;
  sts1(CS(C_TOT_RAYS), 0.0); sts1(CS(C_TOT_STEPS), 0.0); sts1(CS(C_TOT_RHS), 0.0);
  stamp_start(P.counters);

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
          ray_birth(P.cc, mc, P.cc.ray_begin + slot * P.cc.ray_stride, nr, nth, nph, pt, npr, npth, pph);
          nt = 0.0; nlam = 0.0;
          mode = MODE_FRESH;
          n_acc = n_rej = n_cross = n_rec = n_land = 0;
          const double inf = __longlong_as_double(0x7ff0000000000000LL);
          sts1(CS(C_HMAX), 0.0); sts1(CS(C_QDRIFT), 0.0); sts1(CS(C_Q0), 0.0); sts1(CS(C_IQ0), 1.0);
          sts1(CS(C_SINMIN), inf); sts1(CS(C_MARGIN), inf);
        }
      }
    }
    if (!__any_sync(kFull, mode != MODE_IDLE)) break;

    if (mode != MODE_IDLE) {
      // ---- A: F at the pending state (stage 7 of the attempt in flight / k1 of a fresh ray) ----
      Rhs o7;
      rhs_eval<METRIC, true>(mc, pt, pph, nr, nth, npr, npth, o7);

      // ---- B: decisions ----
      bool finished = false;
      bool moved = false;   // y_n changed: run the stop tests' monitor on the new state
      double monH = 0.0, monQ = 0.0, monS = 0.0;
      double lam = 0.0;     // lambda of y_n, valid after this block when mode == MODE_NORMAL
      if (mode == MODE_FRESH) {
        r = nr; th = nth; pr = npr; pth = npth; lam = nlam;
        sts1(CS(C_T), nt); sts1(CS(C_PH), nph); sts1(CS(C_LAM), nlam);
        k1r = o7.dr; k1th = o7.dth; k1pr = o7.dpr; k1pth = o7.dpth;
        sts1(CS(C_K1T), o7.dt); sts1(CS(C_K1PH), o7.dph);
        h = P.h_cap_rel * nr;               // R10 item 4: h0 = cap x the start radius (r_obs for the pinhole)
        monH = fabs(0.5 * o7.H2); monQ = carter_q<METRIC>(mc, pt, pph, npth, o7); monS = fabs(o7.s);
        mode = MODE_NORMAL;
        moved = true;
      } else if (mode == MODE_NORMAL) {
        const double t = lds1(CS(C_T)), ph = lds1(CS(C_PH));
        lam = lds1(CS(C_LAM));
        // R10 items 1-3: scaled max-norm over the six evolving components,
        //   err = max_j |h (e_j + E7 k7_j)| / (atol + rtol max(|y_j|, |y+_j|)).
        // The largest ratio is found by cross-multiplication (num_j den_best > num_best den_j) and
        // divided once; a tie within rounding picks either of two equal ratios.
        // |h| is common to the six numerators and multiplies the winner only; the scale is built as
        // |larger of y, y+| * rtol + atol with the abs folded into the multiply's operand modifier.
#define GP_SCALE(y_, ny_) (__dmul_rn(fabs(fabs(y_) > fabs(ny_) ? (y_) : (ny_)), P.rtol) + P.atol)
        double nm = fabs(et + dp.E7 * o7.dt), dn = GP_SCALE(t, nt);
        double nsum = nm;
#define GP_ERR_TERM(e_, k7_, y_, ny_)                                            \
  {                                                                              \
    double n_ = fabs((e_) + dp.E7 * (k7_));                                      \
    double d_ = GP_SCALE(y_, ny_);                                               \
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
#undef GP_SCALE
        nm *= fabs(h);
        // finite test on the sums: any inf/NaN term makes them non-finite (numerators are >= 0)
        double ysum = ((nt + nr) + (nth + nph)) + (npr + npth);
        double err = div_nr(nm, dn, rcp_nr(dn));
        if (!finite_d(nsum) || !finite_d(ysum) || !finite_d(err)) {
          ++n_rej;
          h *= dp.fac_min;
        } else {
          sts1(CS(C_MARGIN), dmin(lds1(CS(C_MARGIN)), fabs(err - 1.0)));
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
              sts1(CS(C_TARGET), (nr > P.r_esc) ? P.r_esc : P.r_cap);
              mode = MODE_LAND_R;
            } else {
              bool commit = true;
              if ((th - kHalfPi) * (nth - kHalfPi) < 0.0) {
                ++n_cross;
                if (DISK && n_rec < (unsigned)P.max_crossings) {
                  // O7: locate the crossing from y_n; resume from the parked trial state afterwards
                  sts1(PS(0), nr); sts1(PS(1), nth); sts1(PS(2), npr); sts1(PS(3), npth);
                  sts1(PS(4), nt); sts1(PS(5), nph); sts1(PS(6), lam + h); sts1(PS(7), hnext);
                  sts1(PS(8), o7.dt); sts1(PS(9), o7.dr); sts1(PS(10), o7.dth);
                  sts1(PS(11), o7.dph); sts1(PS(12), o7.dpr); sts1(PS(13), o7.dpth);
                  sts1(PS(14), fabs(0.5 * o7.H2));
                  sts1(PS(15), carter_q<METRIC>(mc, pt, pph, npth, o7));
                  sts1(PS(16), fabs(o7.s));
                  sts1(CS(C_TARGET), kHalfPi);
                  mode = MODE_LAND_TH;
                  commit = false;
                }
              }
              if (commit) {
                monH = fabs(0.5 * o7.H2); monQ = carter_q<METRIC>(mc, pt, pph, npth, o7); monS = fabs(o7.s);
                r = nr; th = nth; pr = npr; pth = npth; lam += h;
                sts1(CS(C_T), nt); sts1(CS(C_PH), nph); sts1(CS(C_LAM), lam);
                k1r = o7.dr; k1th = o7.dth; k1pr = o7.dpr; k1pth = o7.dpth;
                sts1(CS(C_K1T), o7.dt); sts1(CS(C_K1PH), o7.dph);
                h = hnext;
                moved = true;
              }
            }
          }
        }
      } else if (mode == MODE_LAND_R) {
        // landed on the exit surface: the record is the landed state (R14)
        r = lds1(CS(C_TARGET)); th = nth; pr = npr; pth = npth;
        sts1(CS(C_T), nt); sts1(CS(C_PH), nph); sts1(CS(C_LAM), nlam);
        ++n_land;
        finished = true;
      } else {  // MODE_LAND_TH
        ++n_land;
        if (DISK) {
          double rc = nr;
          if (rc >= P.disk_r_in && rc <= P.disk_r_out) {
            P.disk[slot].r_cross[n_rec] = rc;
            P.disk[slot].g[n_rec] = kepler_g<METRIC>(mc, rc, pt, pph);
            ++n_rec;
          }
          r = lds1(PS(0)); th = lds1(PS(1)); pr = lds1(PS(2)); pth = lds1(PS(3));
          lam = lds1(PS(6)); h = lds1(PS(7));
          sts1(CS(C_T), lds1(PS(4))); sts1(CS(C_PH), lds1(PS(5))); sts1(CS(C_LAM), lam);
          sts1(CS(C_K1T), lds1(PS(8))); sts1(CS(C_K1PH), lds1(PS(11)));
          k1r = lds1(PS(9)); k1th = lds1(PS(10)); k1pr = lds1(PS(12)); k1pth = lds1(PS(13));
          monH = lds1(PS(14)); monQ = lds1(PS(15)); monS = lds1(PS(16));
        }
        mode = MODE_NORMAL;
        moved = true;
      }

      // stop tests in the oracle's order (R18, R10 item 5), then the monitors of the new state (R22)
      if (mode == MODE_NORMAL) {
        // max_steps <= 5e8 (validated by the host) fits the 32-bit counters; lambda_max is +inf when off
        if (n_acc + n_rej >= (unsigned)P.max_steps || lam >= P.lambda_max) {
          status = GP_RAY_MAXSTEPS;
          finished = true;
        } else if (h < dp.h_floor || h < dp.h_floor * fabs(lam)) {   // h < h_floor max(1, |lambda|)
          status = GP_RAY_STEP_UNDERFLOW;
          finished = true;
        } else if (moved) {
          Monitors mo;
          mo.h_max = lds1(CS(C_HMAX)); mo.q_drift = lds1(CS(C_QDRIFT)); mo.Q0 = lds1(CS(C_Q0));
          mo.iQ0 = lds1(CS(C_IQ0)); mo.sin_min = lds1(CS(C_SINMIN)); mo.err_margin = 0.0;
          monitor_apply<METRIC>(mo, monH, monQ, monS, n_acc == 0 && n_rej == 0);
          sts1(CS(C_HMAX), mo.h_max); sts1(CS(C_SINMIN), mo.sin_min);
          if (METRIC != METRIC_MN) {
            sts1(CS(C_QDRIFT), mo.q_drift); sts1(CS(C_Q0), mo.Q0); sts1(CS(C_IQ0), mo.iQ0);
          }
        }
      }

      if (finished) {
        unsigned attempts = n_acc + n_rej;
        unsigned n_rhs = 1u + 6u * attempts + 5u * n_land;
        Monitors mo;
        mo.h_max = lds1(CS(C_HMAX)); mo.q_drift = lds1(CS(C_QDRIFT)); mo.Q0 = 0.0; mo.iQ0 = 0.0;
        mo.sin_min = lds1(CS(C_SINMIN)); mo.err_margin = lds1(CS(C_MARGIN));
        store_record(P.rays + slot, lds1(CS(C_T)), r, th, lds1(CS(C_PH)), pr, pth, lds1(CS(C_LAM)), pt, pph, mo,
                     status, n_acc, n_rej, n_cross, n_rec, n_rhs);
        if (DISK) {
          const double qnan = __longlong_as_double(0x7ff8000000000000LL);
          for (unsigned i = n_rec; i < 3u; ++i) {
            P.disk[slot].r_cross[i] = qnan;
            P.disk[slot].g[i] = qnan;
          }
        }
        stamp_ray_done(P.counters, P.cc.ray_count);
        sts1(CS(C_TOT_RAYS), lds1(CS(C_TOT_RAYS)) + 1.0);
        sts1(CS(C_TOT_STEPS), lds1(CS(C_TOT_STEPS)) + (double)attempts);
        sts1(CS(C_TOT_RHS), lds1(CS(C_TOT_RHS)) + (double)n_rhs);
        mode = MODE_IDLE;
      } else {
        // ---- C: stages 2..6 of the next attempt from (y_n, k1) ----
        // step and reciprocal selector: ordinary step s = h, divisor 1; landing s = target - y_w,
        // divisor F_w (w = r or theta).  A landing step never returns to (y_n, k1) — the ray ends
        // (r) or resumes from the parked state (theta) — so k1 is scaled in place.
        const bool land_r = (mode == MODE_LAND_R), land_th = (mode == MODE_LAND_TH);
        const bool landing = land_r || land_th;
        // Landing steps are 1 in ~300; the divisor work below is skipped by a warp-uniform branch
        // unless some lane of this convergence group is landing.
        const bool any_land = __any_sync(__activemask(), landing);
        double s = h;
        double bl = 1.0;             // sum of b_i / F_w: d(lambda)/ds of the step, 1 for an ordinary step
        double k1t = lds1(CS(C_K1T)), k1ph = lds1(CS(C_K1PH));
        if (any_land) {
          double iv = 1.0;
          if (landing) {
            s = lds1(CS(C_TARGET)) - (land_r ? r : th);
            iv = rcp_nr(land_r ? k1r : k1th);
          }
          k1r *= iv; k1th *= iv; k1pr *= iv; k1pth *= iv; k1t *= iv; k1ph *= iv;
          bl = dp.B1 * iv;
        }
        // divide the stage slopes of a landing lane by F_w and add its b_i / F_w to bl
#define GP_HENON(b_i)                                                           \
  if (any_land) {                                                               \
    double iv = landing ? rcp_nr(land_r ? o.dr : o.dth) : 1.0;                  \
    o.dr *= iv; o.dth *= iv; o.dpr *= iv; o.dpth *= iv; o.dt *= iv; o.dph *= iv; \
    bl += (b_i) * iv;                                                           \
  }
        // quadratures t, phi: running 5th-order sums and the two error sums
        double bt = dp.B1 * k1t, bph = dp.B1 * k1ph;
        double qet = dp.E1 * k1t, qeph = dp.E1 * k1ph;
        Rhs o;
        double ar, ath, apr, apth;   // K_j of the stage just evaluated
        double br, bth, bpr, bpth;   // K's streamed back from shared memory
        // stage 2
        rhs_eval<METRIC, true>(mc, pt, pph, r + s * (dp.A21 * k1r), th + s * (dp.A21 * k1th),
                         pr + s * (dp.A21 * k1pr), pth + s * (dp.A21 * k1pth), o);
        GP_HENON(0.0)
        ar = o.dr; ath = o.dth; apr = o.dpr; apth = o.dpth;                         // K2
        sts2(KS(0), ar, ath); sts2(KS(1), apr, apth);
        // stage 3
        rhs_eval<METRIC, true>(mc, pt, pph, r + s * (dp.A31 * k1r + dp.A32 * ar),
                         th + s * (dp.A31 * k1th + dp.A32 * ath),
                         pr + s * (dp.A31 * k1pr + dp.A32 * apr),
                         pth + s * (dp.A31 * k1pth + dp.A32 * apth), o);
        GP_HENON(dp.B3)
        ar = o.dr; ath = o.dth; apr = o.dpr; apth = o.dpth;                         // K3
        sts2(KS(2), ar, ath); sts2(KS(3), apr, apth);
        bt += dp.B3 * o.dt; bph += dp.B3 * o.dph;
        qet += dp.E3 * o.dt; qeph += dp.E3 * o.dph;
        // stage 4
        {
          double xr = dp.A41 * k1r + dp.A43 * ar, xth = dp.A41 * k1th + dp.A43 * ath;
          double xpr = dp.A41 * k1pr + dp.A43 * apr, xpth = dp.A41 * k1pth + dp.A43 * apth;
          lds2(KS(0), br, bth); lds2(KS(1), bpr, bpth);                             // K2
          xr += dp.A42 * br; xth += dp.A42 * bth; xpr += dp.A42 * bpr; xpth += dp.A42 * bpth;
          rhs_eval<METRIC, true>(mc, pt, pph, r + s * xr, th + s * xth, pr + s * xpr, pth + s * xpth, o);
        }
        GP_HENON(dp.B4)
        ar = o.dr; ath = o.dth; apr = o.dpr; apth = o.dpth;                         // K4
        sts2(KS(4), ar, ath); sts2(KS(5), apr, apth);
        bt += dp.B4 * o.dt; bph += dp.B4 * o.dph;
        qet += dp.E4 * o.dt; qeph += dp.E4 * o.dph;
        // stage 5
        {
          double xr = dp.A51 * k1r + dp.A54 * ar, xth = dp.A51 * k1th + dp.A54 * ath;
          double xpr = dp.A51 * k1pr + dp.A54 * apr, xpth = dp.A51 * k1pth + dp.A54 * apth;
          lds2(KS(0), br, bth); lds2(KS(1), bpr, bpth);                             // K2
          xr += dp.A52 * br; xth += dp.A52 * bth; xpr += dp.A52 * bpr; xpth += dp.A52 * bpth;
          lds2(KS(2), br, bth); lds2(KS(3), bpr, bpth);                             // K3
          xr += dp.A53 * br; xth += dp.A53 * bth; xpr += dp.A53 * bpr; xpth += dp.A53 * bpth;
          rhs_eval<METRIC, true>(mc, pt, pph, r + s * xr, th + s * xth, pr + s * xpr, pth + s * xpth, o);
        }
        GP_HENON(dp.B5)
        ar = o.dr; ath = o.dth; apr = o.dpr; apth = o.dpth;                         // K5
        sts2(KS(6), ar, ath); sts2(KS(7), apr, apth);
        bt += dp.B5 * o.dt; bph += dp.B5 * o.dph;
        qet += dp.E5 * o.dt; qeph += dp.E5 * o.dph;
        // stage 6
        {
          double xr = dp.A61 * k1r + dp.A65 * ar, xth = dp.A61 * k1th + dp.A65 * ath;
          double xpr = dp.A61 * k1pr + dp.A65 * apr, xpth = dp.A61 * k1pth + dp.A65 * apth;
          lds2(KS(0), br, bth); lds2(KS(1), bpr, bpth);                             // K2
          xr += dp.A62 * br; xth += dp.A62 * bth; xpr += dp.A62 * bpr; xpth += dp.A62 * bpth;
          lds2(KS(2), br, bth); lds2(KS(3), bpr, bpth);                             // K3
          xr += dp.A63 * br; xth += dp.A63 * bth; xpr += dp.A63 * bpr; xpth += dp.A63 * bpth;
          lds2(KS(4), br, bth); lds2(KS(5), bpr, bpth);                             // K4
          xr += dp.A64 * br; xth += dp.A64 * bth; xpr += dp.A64 * bpr; xpth += dp.A64 * bpth;
          rhs_eval<METRIC, true>(mc, pt, pph, r + s * xr, th + s * xth, pr + s * xpr, pth + s * xpth, o);
        }
        GP_HENON(dp.B6)
        ar = o.dr; ath = o.dth; apr = o.dpr; apth = o.dpth;                         // K6
        bt += dp.B6 * o.dt; bph += dp.B6 * o.dph;
        qet += dp.E6 * o.dt; qeph += dp.E6 * o.dph;
#undef GP_HENON
        // trial end state (5th-order solution; a7 = b) and the error sums without e7 k7
        {
          double xr = dp.B1 * k1r + dp.B6 * ar, xth = dp.B1 * k1th + dp.B6 * ath;
          double xpr = dp.B1 * k1pr + dp.B6 * apr, xpth = dp.B1 * k1pth + dp.B6 * apth;
          er = dp.E1 * k1r + dp.E6 * ar; eth = dp.E1 * k1th + dp.E6 * ath;
          epr = dp.E1 * k1pr + dp.E6 * apr; epth = dp.E1 * k1pth + dp.E6 * apth;
          lds2(KS(2), br, bth); lds2(KS(3), bpr, bpth);                             // K3
          xr += dp.B3 * br; xth += dp.B3 * bth; xpr += dp.B3 * bpr; xpth += dp.B3 * bpth;
          er += dp.E3 * br; eth += dp.E3 * bth; epr += dp.E3 * bpr; epth += dp.E3 * bpth;
          lds2(KS(4), br, bth); lds2(KS(5), bpr, bpth);                             // K4
          xr += dp.B4 * br; xth += dp.B4 * bth; xpr += dp.B4 * bpr; xpth += dp.B4 * bpth;
          er += dp.E4 * br; eth += dp.E4 * bth; epr += dp.E4 * bpr; epth += dp.E4 * bpth;
          lds2(KS(6), br, bth); lds2(KS(7), bpr, bpth);                             // K5
          xr += dp.B5 * br; xth += dp.B5 * bth; xpr += dp.B5 * bpr; xpth += dp.B5 * bpth;
          er += dp.E5 * br; eth += dp.E5 * bth; epr += dp.E5 * bpr; epth += dp.E5 * bpth;
          nr = r + s * xr; nth = th + s * xth; npr = pr + s * xpr; npth = pth + s * xpth;
        }
        nt = lds1(CS(C_T)) + s * bt;
        nph = lds1(CS(C_PH)) + s * bph;
        nlam = lds1(CS(C_LAM)) + s * bl;
        et = qet;
        eph = qeph;
      }
    }
  }

  // totals (gp.h: counters[1] rays finished, [2] attempted steps, [3] RHS evaluations)
  {
    const double tr = lds1(CS(C_TOT_RAYS));
    if (tr > 0.0) {
      atomicAdd(P.counters + 1, (unsigned long long)tr);
      atomicAdd(P.counters + 2, (unsigned long long)lds1(CS(C_TOT_STEPS)));
      atomicAdd(P.counters + 3, (unsigned long long)lds1(CS(C_TOT_RHS)));
    }
  }
  stamp_end(P.counters);
#undef KS
#undef CS
#undef PS
}

#endif  // __CUDACC__
}  // namespace gp
#endif
