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
// touches; the rest lives in shared memory so that four blocks (16 warps) fit per SM in 128 registers.
// Everything is laid out [pair][lane], 16 bytes per lane, behind ONE per-lane base address:
//   K area   11 x double2  stage slopes K2..K5 of (r, th) and (p_r, p_th) (pairs 0-7), the RAW k1 = F(y_n)
//                          of the same four components (pairs 8, 9; read once per attempt, so that a
//                          rejected step retries from it) and (sin, cos) theta_n (pair 10).  128-bit
//                          accesses, conflict-free.
//   cold     kColdSlots x double (two per pair)   state the stages never read: t, phi, lambda, the monitors,
//                          the landing target, k1 of the two quadratures, the per-lane totals, the output
//                          slot, the rare counters, status, segment start.
//   park     8 x double    (disk and ring variants) what a ray resumes from after a landing step located
//                          something on the way: the accepted trial state (r, th, pr, pth, t, ph, lambda) and
//                          the next step.  F there is evaluated again when the ray resumes (MODE_RESUME: one
//                          evaluation per landing, the same bits) instead of being parked with its monitor
//                          triple: 17 doubles made the block 60 KB and held these variants to three blocks per
//                          SM; with 8 it is 50 KB and four fit, like the headline kernel.
enum { C_T = 0, C_PH, C_LAM, C_HMAX, C_QDRIFT, C_Q0, C_IQ0, C_SINMIN, C_MARGIN, C_TARGET, C_K1T, C_K1PH,
       C_TOT_RAYS, C_TOT_STEPS, C_TOT_RHS,
       C_SLOT,      // output slot of the ray in flight (64-bit integer bits)
       C_COUNTS,    // n_equator_crossings (low word) and landing steps taken (high word)
       C_STATE,     // status of the ray once decided (low word) and disk crossings recorded (high word)
       C_SEG,       // attempted steps at the start of this segment (segmented tracing)
       C_NREJ,      // rejected steps (touched on a rejection only; a register holds the attempts)
       kColdSlots };
constexpr int kKSlots2 = 11;   // + (sin, cos) of theta_n
constexpr int kParkSlotsDp54 = 8;
// Every area is laid out [pair][lane] with 16 bytes per lane, so that ONE per-lane base address (plus
// compile-time offsets) reaches everything: a double slot j of the cold or park area is half (j & 1) of
// pair j / 2.  (With separate 8- and 16-byte strides the compiler rebuilt two or three base addresses from
// %tid and the shared window several times per step.)
constexpr int kColdPairs = (kColdSlots + 1) / 2, kParkPairs = (kParkSlotsDp54 + 1) / 2;
constexpr size_t dp54_smem_bytes(bool parked) {
  return 16 * (size_t)kBlock * (kKSlots2 + kColdPairs + (parked ? kParkPairs : 0));
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

// OBJ: 0 no object; 1 thin disk, crossings located and recorded (R19); 2 solid ring, the ray ends where it
// enters the volume (R39).  Both objects use the park area.
// TR: arithmetic type of Hamilton's equations.  double is the required path; float is the mixed variant
// (cfg.precision = 2): FP32 equations at the rounded state, FP64 state, sums, error
// norm and controller — the tolerance must then stay above the noise of an FP32 evaluation (gp.h).
template <int METRIC, int OBJ, class TR = double>
__global__ void __launch_bounds__(kBlock, METRIC == METRIC_MN ? GP_DP54_MIN_BLOCKS_MN : GP_DP54_MIN_BLOCKS)
trace_dp54(const __grid_constant__ TraceParams P) {
  constexpr bool DISK = (OBJ == 1), RING = (OBJ == 2), MIXED = (sizeof(TR) == 4);
  constexpr bool SEG = (METRIC == METRIC_MN);   // segmented tracing is built into the Manko-Novikov kernels only
  extern __shared__ double2 smem2[];
  const MetricConst &mc = P.mc;
  const int tid = threadIdx.x;
  // the one per-lane base address, produced by an asm volatile so that ptxas keeps it in a register
  // instead of rebuilding it from %tid and the shared window two or three times per step
  unsigned sm_k;
  asm volatile("mad.lo.u32 %0, %1, 16, %2;" : "=r"(sm_k) : "r"(tid), "r"((unsigned)__cvta_generic_to_shared(smem2)));
#define KS(slot) (sm_k + 16u * kBlock * (slot))
#define CS(slot) (sm_k + 16u * kBlock * (kKSlots2 + (slot) / 2) + 8u * ((slot) & 1))
#define PS(slot) (sm_k + 16u * kBlock * (kKSlots2 + kColdPairs + (slot) / 2) + 8u * ((slot) & 1))

  // ---- per-lane ray state (registers) ----
  int mode = MODE_IDLE;
  double pt = 0.0, pph = 0.0;                         // constants of the ray
  double r = 0.0, th = 0.0, pr = 0.0, pth = 0.0;      // y_n, the part Hamilton's equations read
  // raw F(y_n) lives in shared memory (K slots 8, 9): written when y_n changes, read once per attempt
#define GP_SET_K1(a_, b_, c_, d_) { sts2(KS(8), (a_), (b_)); sts2(KS(9), (c_), (d_)); }
#define GP_SET_SC(s_, c_) if (METRIC == METRIC_KERR && !MIXED) sts2(KS(10), (s_), (c_));
  double h = 0.0;                                     // step of the attempt in flight / next attempt
  // pending (trial) state and the error sums that still lack the e7 k7 term
  double nt = 0.0, nr = 0.0, nth = 0.0, nph = 0.0, npr = 0.0, npth = 0.0, nlam = 0.0;
  double et = 0.0, er = 0.0, eth = 0.0, eph = 0.0, epr = 0.0, epth = 0.0;
  unsigned n_att = 0;   // attempted steps; n_rej: cold slot C_NREJ; n_cross, n_land: C_COUNTS; status, n_rec: C_STATE
#define GP_BUMP_REJ() sts1(CS(C_NREJ), __hiloint2double(0, __double2loint(lds1(CS(C_NREJ))) + 1));
#define GP_SET_STATUS(code_)                                                                   \
  {                                                                                            \
    double w_ = lds1(CS(C_STATE));                                                             \
    sts1(CS(C_STATE), __hiloint2double(__double2hiint(w_), (int)(code_)));                     \
  }
// the ray goes on from the trial state parked before a landing step (thin disk: always; ring: no hit);
// the ring variant counts the equator crossing of that step here (the oracle counts it after its ring test)
#define GP_RESUME_PARKED()                                                                     \
  {                                                                                            \
    if (RING && (th - kHalfPi) * (lds1(PS(1)) - kHalfPi) < 0.0) GP_BUMP_COUNTS(1, 0)           \
    nr = lds1(PS(0)); nth = lds1(PS(1)); npr = lds1(PS(2)); npth = lds1(PS(3));                \
    nt = lds1(PS(4)); nph = lds1(PS(5)); nlam = lds1(PS(6)); h = lds1(PS(7));                  \
    mode = MODE_RESUME;   /* block A of the next trip evaluates F there, block B takes it as y_n */ \
  }
#define GP_BUMP_COUNTS(dcross_, dland_)                                                        \
  {                                                                                            \
    double w_ = lds1(CS(C_COUNTS));                                                            \
    sts1(CS(C_COUNTS), __hiloint2double(__double2hiint(w_) + (dland_), __double2loint(w_) + (dcross_))); \
  }
  bool exhausted = false;
  sts1(CS(C_TOT_RAYS), 0.0); sts1(CS(C_TOT_STEPS), 0.0); sts1(CS(C_TOT_RHS), 0.0);
  stamp_start(P.counters);

  for (;;) {
    // ---- a1: refill idle lanes ----
    const bool need = (mode == MODE_IDLE) && !exhausted;
    const unsigned need_mask = __ballot_sync(kFull, need);
    if (need_mask) {
      const bool from_list = SEG && P.round > 0;
      const long long n_work = from_list ? (long long)*P.list_in_count : P.cc.ray_count;
      const long long got = fetch_slot(need_mask, need, P.counters, n_work);
      if (need) {
        const long long slot = (from_list && got >= 0) ? P.list_in[got] : got;
        if (slot < 0) {
          exhausted = true;
        } else if (from_list) {
          // resume a parked ray: its record holds y_n, the constants, the monitors and the counters; the
          // step proposal sits in the q_drift field (unused by this metric) and the landing-step count in
          // n_rhs.  F(y_n) is evaluated afresh in block A — the same bits the FSAL evaluation had.
          const double *rec = reinterpret_cast<const double *>(P.rays + slot);
          nt = rec[0]; nr = rec[1]; nth = rec[2]; nph = rec[3];
          nlam = rec[4]; npr = rec[6]; npth = rec[7];
          pt = rec[8]; pph = rec[9];
          h = rec[11];
          const double w0 = rec[5], w1 = rec[14], w2 = rec[15];
          n_att = (unsigned)__double2hiint(w0) + (unsigned)__double2loint(w1);
          sts1(CS(C_NREJ), __hiloint2double(0, __double2loint(w1)));
          sts1(CS(C_HMAX), rec[10]); sts1(CS(C_QDRIFT), 0.0); sts1(CS(C_Q0), 0.0); sts1(CS(C_IQ0), 1.0);
          sts1(CS(C_SINMIN), rec[12]); sts1(CS(C_MARGIN), rec[13]);
          sts1(CS(C_SLOT), __longlong_as_double(slot));
          sts1(CS(C_COUNTS), __hiloint2double(__double2hiint(w2), __double2hiint(w1)));   // n_land | n_cross
          sts1(CS(C_STATE), __hiloint2double(__double2loint(w2), 0));                      // n_rec | status
          sts1(CS(C_SEG), (double)n_att);
          mode = MODE_RESUME;
        } else {
          // a2 + a3
          ray_birth(P.cc, mc, P.cc.ray_begin + slot * P.cc.ray_stride, nr, nth, nph, pt, npr, npth, pph);
          nt = 0.0; nlam = 0.0;
          mode = MODE_FRESH;
          n_att = 0;
          sts1(CS(C_NREJ), __longlong_as_double(0LL));
          sts1(CS(C_SLOT), __longlong_as_double(slot)); sts1(CS(C_COUNTS), __longlong_as_double(0LL));
          sts1(CS(C_STATE), __longlong_as_double(0LL));
          if (SEG) sts1(CS(C_SEG), 0.0);
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
      if (MIXED) rhs_eval_fp32_scaled<METRIC>(mc, pt, pph, nr, nth, npr, npth, 1.0, o7);
      else rhs_eval<METRIC, true>(mc, pt, pph, nr, nth, npr, npth, o7);

      // ---- B: decisions ----
      bool finished = false;
      bool moved = false;   // y_n changed: run the stop tests' monitor on the new state
      double monH = 0.0, monQ = 0.0, monS = 0.0;
      double lam = 0.0;     // lambda of y_n, valid after this block when mode == MODE_NORMAL
      constexpr bool kResumes = SEG || OBJ != 0;   // MODE_RESUME exists: segmented tracing, or a parked trial state
      if (mode == MODE_FRESH || (kResumes && mode == MODE_RESUME)) {
        r = nr; th = nth; pr = npr; pth = npth; lam = nlam;
        sts1(CS(C_T), nt); sts1(CS(C_PH), nph); sts1(CS(C_LAM), nlam);
        GP_SET_K1(o7.dr, o7.dth, o7.dpr, o7.dpth)
        GP_SET_SC(o7.s, o7.c)
        sts1(CS(C_K1T), o7.dt); sts1(CS(C_K1PH), o7.dph);
        if (!kResumes || mode == MODE_FRESH) h = P.h_cap_rel * nr;   // R10 item 4: h0 = cap x the start radius (r_obs for the pinhole); a resumed ray keeps its proposal
        monH = fabs(0.5 * o7.H2); monQ = carter_q<METRIC>(mc, pt, pph, npth, o7); monS = fabs(o7.s);
        if (METRIC != METRIC_MN && mode == MODE_FRESH) {
          // the reference value of the Carter monitor (R23) is set here, once per ray, so that the per-step
          // monitor below carries no "first step" instructions
          sts1(CS(C_Q0), monQ);
          sts1(CS(C_IQ0), rcp_nr(dmax(1.0, fabs(monQ))));
        }
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
#define GP_SCALE(y_, ny_) fma(fabs(fabs(y_) > fabs(ny_) ? (y_) : (ny_)), P.rtol, P.atol)
        const double hE7 = dp.E7 * h;     // the error sums already carry the step (block C)
        double nm = fabs(et + hE7 * o7.dt), dn = GP_SCALE(t, nt);
        double nsum = nm;
#define GP_ERR_TERM(e_, k7_, y_, ny_)                                            \
  {                                                                              \
    double n_ = fabs((e_) + hE7 * (k7_));                                        \
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
        // finite test on the sums: any inf/NaN term makes them non-finite (numerators are >= 0)
        double err = div_nr(nm, dn, rcp_nr(dn));
        // R10 item 2: a non-finite estimate or trial state is a rejection with the factor 0.2.  The two kinds of
        // rejection share one (rare) block, so that neither is if-converted into predicated instructions that
        // every step would issue.
        const bool bad = !finite_d(nsum) || !finite_d(err);
        if (!bad) sts1(CS(C_MARGIN), dmin(lds1(CS(C_MARGIN)), fabs(err - 1.0)));
        // fac = 0.9 err^(-1/5), clamped to [0.2, 5] (err = 0 gives 5); the range clamp sits on the FP32 seed
        // of the fifth root and changes nothing: 0.9 (1e-5)^-0.2 = 9 > 5, 0.9 (1e4)^-0.2 = 0.14 < 0.2
        double fac = dp.safety * pow_m1_5_clamped(err);
        fac = dmin(dmax(dp.fac_min, fac), 5.0);   // R10 item 3 (5.0 as an immediate)
        ++n_att;
        {
          if (bad || err > 1.0) {
            GP_BUMP_REJ()
            h *= bad ? dp.fac_min : fac;
          } else {
            double hnext = dmin(h * fac, P.h_cap_rel * nr);
            if (nr > P.r_esc || nr < P.r_cap) {
              // O8: discard the step, land on the surface from y_n
              GP_SET_STATUS((nr > P.r_esc) ? GP_RAY_ESCAPED : GP_RAY_CAPTURED)
              sts1(CS(C_TARGET), (nr > P.r_esc) ? P.r_esc : P.r_cap);
              mode = MODE_LAND_R;
            } else {
              bool commit = true;
              // park the accepted trial state and the next step, so that the ray can resume from it after a
              // landing step located something on the way from y_n
#define GP_PARK()                                                                        \
  {                                                                                      \
    sts1(PS(0), nr); sts1(PS(1), nth); sts1(PS(2), npr); sts1(PS(3), npth);              \
    sts1(PS(4), nt); sts1(PS(5), nph); sts1(PS(6), lam + h); sts1(PS(7), hnext);         \
  }
              bool ring_try = false;
              if (RING) {
                // R39: the step can meet the box r_in..r_out x |theta - pi/2| <= d only if every coordinate
                // that starts outside its interval ends inside it or beyond it
                const double un = th - kHalfPi, un1 = nth - kHalfPi;
                const bool th_out = fabs(un) > P.ring_d;
                const bool r_out_n = !(r >= P.disk_r_in && r <= P.disk_r_out);
                const bool th_enters = fabs(un1) <= P.ring_d || un * un1 < 0.0;
                const bool r_enters = (nr >= P.disk_r_in && nr <= P.disk_r_out) || ((r < P.disk_r_in) != (nr < P.disk_r_in));
                ring_try = (th_out || r_out_n) && (!th_out || th_enters) && (!r_out_n || r_enters);
                if (ring_try) {
                  GP_PARK()
                  if (th_out) {
                    sts1(CS(C_TARGET), kHalfPi + (un > 0.0 ? P.ring_d : -P.ring_d));
                    mode = MODE_LAND_TH;
                  } else {
                    GP_SET_STATUS(GP_RAY_HIT_RING)
                    sts1(CS(C_TARGET), (r < P.disk_r_in) ? P.disk_r_in : P.disk_r_out);
                    mode = MODE_LAND_R;
                  }
                  commit = false;
                }
              }
              // (ring variant: a step under examination counts its equator crossing when it resumes)
              if (!ring_try && (th - kHalfPi) * (nth - kHalfPi) < 0.0) {
                GP_BUMP_COUNTS(1, 0)
                if (DISK && (unsigned)__double2hiint(lds1(CS(C_STATE))) < (unsigned)P.max_crossings) {
                  // O7: locate the crossing from y_n; resume from the parked trial state afterwards
                  GP_PARK()
                  sts1(CS(C_TARGET), kHalfPi);
                  mode = MODE_LAND_TH;
                  commit = false;
                }
              }
#undef GP_PARK
              if (commit) {
                monH = fabs(0.5 * o7.H2); monQ = carter_q<METRIC>(mc, pt, pph, npth, o7); monS = fabs(o7.s);
                r = nr; th = nth; pr = npr; pth = npth; lam += h;
                sts1(CS(C_T), nt); sts1(CS(C_PH), nph); sts1(CS(C_LAM), lam);
                GP_SET_K1(o7.dr, o7.dth, o7.dpr, o7.dpth)
                GP_SET_SC(o7.s, o7.c)
                sts1(CS(C_K1T), o7.dt); sts1(CS(C_K1PH), o7.dph);
                h = hnext;
                moved = true;
              }
            }
          }
        }
      } else if (mode == MODE_LAND_R) {
        GP_BUMP_COUNTS(0, 1)
        bool resume = false;
        if (RING && __double2loint(lds1(CS(C_STATE))) == GP_RAY_HIT_RING) {
          // radial face of the ring: a hit if the landed theta is inside the slab, else the ray goes on
          if (fabs(nth - kHalfPi) <= P.ring_d) {
            const long long slot = __double_as_longlong(lds1(CS(C_SLOT)));
            const double rc = lds1(CS(C_TARGET));
            P.disk[slot].r_cross[0] = rc;
            P.disk[slot].g[0] = kepler_g<METRIC>(mc, rc, pt, pph);
            sts1(CS(C_STATE), __hiloint2double(1, GP_RAY_HIT_RING));
          } else {
            GP_SET_STATUS(0)
            resume = true;
          }
        }
        if (!resume) {
          // landed on the exit surface (or the ring's radial face): the record is the landed state (R14)
          r = lds1(CS(C_TARGET)); th = nth; pr = npr; pth = npth;
          sts1(CS(C_T), nt); sts1(CS(C_PH), nph); sts1(CS(C_LAM), nlam);
          finished = true;
        } else {
          GP_RESUME_PARKED()
        }
      } else {  // MODE_LAND_TH
        GP_BUMP_COUNTS(0, 1)
        if (RING) {
          // theta-face of the ring: a hit if the landed radius is in range; else try the radial face on
          // y_n's side when r_n is outside the range; else the ray goes on from the parked state
          if (nr >= P.disk_r_in && nr <= P.disk_r_out) {
            const long long slot = __double_as_longlong(lds1(CS(C_SLOT)));
            P.disk[slot].r_cross[0] = nr;
            P.disk[slot].g[0] = kepler_g<METRIC>(mc, nr, pt, pph);
            sts1(CS(C_STATE), __hiloint2double(1, GP_RAY_HIT_RING));
            r = nr; th = lds1(CS(C_TARGET)); pr = npr; pth = npth;
            sts1(CS(C_T), nt); sts1(CS(C_PH), nph); sts1(CS(C_LAM), nlam);
            finished = true;
          } else if (!(r >= P.disk_r_in && r <= P.disk_r_out)) {
            GP_SET_STATUS(GP_RAY_HIT_RING)
            sts1(CS(C_TARGET), (r < P.disk_r_in) ? P.disk_r_in : P.disk_r_out);
            mode = MODE_LAND_R;
          } else {
            GP_RESUME_PARKED()
          }
        }
        if (DISK) {
          double rc = nr;
          if (rc >= P.disk_r_in && rc <= P.disk_r_out) {
            const long long slot = __double_as_longlong(lds1(CS(C_SLOT)));
            const double sw = lds1(CS(C_STATE));
            const unsigned n_rec = (unsigned)__double2hiint(sw);
            P.disk[slot].r_cross[n_rec] = rc;
            P.disk[slot].g[n_rec] = kepler_g<METRIC>(mc, rc, pt, pph);
            sts1(CS(C_STATE), __hiloint2double((int)(n_rec + 1u), __double2loint(sw)));
          }
          GP_RESUME_PARKED()
        }
        if (OBJ == 0) {
          mode = MODE_NORMAL;
          moved = true;
        }
      }

      // stop tests in the oracle's order (R18, R10 item 5), then the monitors of the new state (R22)
      if (mode == MODE_NORMAL) {
        // max_steps <= 5e8 (validated by the host) fits the 32-bit counters; lambda_max is +inf when off
        const bool budget = n_att >= (unsigned)P.max_steps || lam >= P.lambda_max;
        const bool underflow = h < dp.h_floor * dmax(1.0, fabs(lam));   // R10 item 5 (compare + select, no fmax)
        if (budget || underflow) {            // one rare block for both
          GP_SET_STATUS(budget ? GP_RAY_MAXSTEPS : GP_RAY_STEP_UNDERFLOW)
          finished = true;
        } else if (moved) {
          Monitors mo;
          mo.h_max = lds1(CS(C_HMAX)); mo.q_drift = lds1(CS(C_QDRIFT)); mo.Q0 = lds1(CS(C_Q0));
          mo.iQ0 = lds1(CS(C_IQ0)); mo.sin_min = lds1(CS(C_SINMIN)); mo.err_margin = 0.0;
          monitor_apply<METRIC>(mo, monH, monQ, monS, false);
          sts1(CS(C_HMAX), mo.h_max); sts1(CS(C_SINMIN), mo.sin_min);
          if (METRIC != METRIC_MN) sts1(CS(C_QDRIFT), mo.q_drift);
        }
        // Segmented tracing: a ray that has used up its segment parks (y_n, constants, monitors, counters, step
        // proposal) in its own record and hands its slot to the next round; any lane picks it up there.
        if (SEG && P.seg_steps > 0 && !finished &&
            (long long)n_att - (long long)lds1(CS(C_SEG)) >= P.seg_steps) {
          const unsigned n_rej = (unsigned)__double2loint(lds1(CS(C_NREJ))), n_acc = n_att - n_rej;
          const long long slot = __double_as_longlong(lds1(CS(C_SLOT)));
          const double cw = lds1(CS(C_COUNTS)), sw = lds1(CS(C_STATE));
          Monitors mo;
          mo.h_max = lds1(CS(C_HMAX)); mo.q_drift = h; mo.Q0 = 0.0; mo.iQ0 = 0.0;
          mo.sin_min = lds1(CS(C_SINMIN)); mo.err_margin = lds1(CS(C_MARGIN));
          store_record(P.rays + slot, lds1(CS(C_T)), r, th, lds1(CS(C_PH)), pr, pth, lam, pt, pph, mo, kRayParked,
                       n_acc, n_rej, (unsigned)__double2loint(cw), (unsigned)__double2hiint(sw),
                       (unsigned)__double2hiint(cw));
          P.list_out[atomicAdd(P.list_out_count, 1ull)] = slot;
          mode = MODE_IDLE;
        }
      }

      if (finished) {
        const unsigned attempts = n_att;
        const unsigned n_rej = (unsigned)__double2loint(lds1(CS(C_NREJ))), n_acc = n_att - n_rej;
        const long long slot = __double_as_longlong(lds1(CS(C_SLOT)));
        const double cw = lds1(CS(C_COUNTS));
        const unsigned n_cross = (unsigned)__double2loint(cw), n_land = (unsigned)__double2hiint(cw);
        const double sw = lds1(CS(C_STATE));
        const unsigned status = (unsigned)__double2loint(sw), n_rec = (unsigned)__double2hiint(sw);
        unsigned n_rhs = 1u + 6u * attempts + 5u * n_land;
        Monitors mo;
        mo.h_max = lds1(CS(C_HMAX)); mo.q_drift = lds1(CS(C_QDRIFT)); mo.Q0 = 0.0; mo.iQ0 = 0.0;
        mo.sin_min = lds1(CS(C_SINMIN)); mo.err_margin = lds1(CS(C_MARGIN));
        store_record(P.rays + slot, lds1(CS(C_T)), r, th, lds1(CS(C_PH)), pr, pth, lds1(CS(C_LAM)), pt, pph, mo,
                     status, n_acc, n_rej, n_cross, n_rec, n_rhs);
        if (OBJ != 0) {
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
      } else if (!kResumes || (mode != MODE_IDLE && mode != MODE_RESUME)) {
        // ---- C: stages 2..6 of the next attempt from (y_n, k1) ----
        // (a lane that has just parked its segment, or that resumes from a parked trial state and has no k1
        // yet, sits this block out)
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
        double k1r, k1th, k1pr, k1pth;
        lds2(KS(8), k1r, k1th); lds2(KS(9), k1pr, k1pth);
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
    double iv = landing ? s * rcp_nr(land_r ? o.dr : o.dth) : 1.0;  /* o is s F */ \
    o.dr *= iv; o.dth *= iv; o.dpr *= iv; o.dpth *= iv; o.dt *= iv; o.dph *= iv; \
    bl += (b_i) * iv;                                                           \
  }
        // Every K below is s F (or s F / F_w on a landing lane): the stage evaluations return their
        // derivatives already multiplied by the step (rhs_eval_scaled), k1 is scaled once here, and the
        // stage states, the trial state and the error sums are plain FMA chains from y_n.
        const double hk1r = s * k1r, hk1th = s * k1th, hk1pr = s * k1pr, hk1pth = s * k1pth;
        const double hk1t = s * k1t, hk1ph = s * k1ph;
        // Stage angles (Kerr; for Schwarzschild the extra registers cost a spill): the theta sums below start from 0 instead of theta_n, so they
        // are the increments d_j, and sin, cos of theta_n + d_j come from (sin, cos) theta_n — by-products of
        // the evaluation that produced k1, kept in K slot 10 — through the addition theorems (sincos_add):
        // no range reduction or quadrant logic inside the stages.  Manko-Novikov evaluates its own sincos.
        constexpr bool kAngle = (METRIC == METRIC_KERR) && !MIXED;
        const double thb = kAngle ? 0.0 : th;
        double sn_ = 0.0, cn_ = 0.0;
        if (kAngle) lds2(KS(10), sn_, cn_);
#define GP_STAGE_RHS(xr_, xth_, xpr_, xpth_)                                                   \
  if (kAngle) {                                                                                \
    double ss_, cc_;                                                                           \
    sincos_add(sn_, cn_, (xth_), &ss_, &cc_);                                                  \
    rhs_eval_scaled_sc<METRIC>(mc, pt, pph, (xr_), ss_, cc_, (xpr_), (xpth_), s, o);           \
  } else if (MIXED) {                                                                          \
    rhs_eval_fp32_scaled<METRIC>(mc, pt, pph, (xr_), (xth_), (xpr_), (xpth_), s, o);           \
  } else {                                                                                     \
    rhs_eval_scaled<METRIC, true>(mc, pt, pph, (xr_), (xth_), (xpr_), (xpth_), s, o);          \
  }
        double bt = dp.B1 * hk1t, bph = dp.B1 * hk1ph;
        double qet = dp.E1 * hk1t, qeph = dp.E1 * hk1ph;
        Rhs o;
        double ar, ath, apr, apth;   // K_j of the stage just evaluated
        double br, bth, bpr, bpth;   // K's streamed back from shared memory
        // stage 2
        GP_STAGE_RHS( fma(dp.A21, hk1r, r), fma(dp.A21, hk1th, thb),
                                      fma(dp.A21, hk1pr, pr), fma(dp.A21, hk1pth, pth))
        GP_HENON(0.0)
        ar = o.dr; ath = o.dth; apr = o.dpr; apth = o.dpth;                         // K2
        sts2(KS(0), ar, ath); sts2(KS(1), apr, apth);
        // stage 3
        GP_STAGE_RHS( fma(dp.A32, ar, fma(dp.A31, hk1r, r)),
                                      fma(dp.A32, ath, fma(dp.A31, hk1th, thb)),
                                      fma(dp.A32, apr, fma(dp.A31, hk1pr, pr)),
                                      fma(dp.A32, apth, fma(dp.A31, hk1pth, pth)))
        GP_HENON(dp.B3)
        ar = o.dr; ath = o.dth; apr = o.dpr; apth = o.dpth;                         // K3
        sts2(KS(2), ar, ath); sts2(KS(3), apr, apth);
        bt += dp.B3 * o.dt; bph += dp.B3 * o.dph;
        qet += dp.E3 * o.dt; qeph += dp.E3 * o.dph;
        // stage 4
        {
          double xr = fma(dp.A43, ar, fma(dp.A41, hk1r, r)), xth = fma(dp.A43, ath, fma(dp.A41, hk1th, thb));
          double xpr = fma(dp.A43, apr, fma(dp.A41, hk1pr, pr)), xpth = fma(dp.A43, apth, fma(dp.A41, hk1pth, pth));
          lds2(KS(0), br, bth); lds2(KS(1), bpr, bpth);                             // K2
          xr = fma(dp.A42, br, xr); xth = fma(dp.A42, bth, xth); xpr = fma(dp.A42, bpr, xpr); xpth = fma(dp.A42, bpth, xpth);
          GP_STAGE_RHS( xr, xth, xpr, xpth)
        }
        GP_HENON(dp.B4)
        ar = o.dr; ath = o.dth; apr = o.dpr; apth = o.dpth;                         // K4
        sts2(KS(4), ar, ath); sts2(KS(5), apr, apth);
        bt += dp.B4 * o.dt; bph += dp.B4 * o.dph;
        qet += dp.E4 * o.dt; qeph += dp.E4 * o.dph;
        // stage 5
        {
          double xr = fma(dp.A54, ar, fma(dp.A51, hk1r, r)), xth = fma(dp.A54, ath, fma(dp.A51, hk1th, thb));
          double xpr = fma(dp.A54, apr, fma(dp.A51, hk1pr, pr)), xpth = fma(dp.A54, apth, fma(dp.A51, hk1pth, pth));
          lds2(KS(0), br, bth); lds2(KS(1), bpr, bpth);                             // K2
          xr = fma(dp.A52, br, xr); xth = fma(dp.A52, bth, xth); xpr = fma(dp.A52, bpr, xpr); xpth = fma(dp.A52, bpth, xpth);
          lds2(KS(2), br, bth); lds2(KS(3), bpr, bpth);                             // K3
          xr = fma(dp.A53, br, xr); xth = fma(dp.A53, bth, xth); xpr = fma(dp.A53, bpr, xpr); xpth = fma(dp.A53, bpth, xpth);
          GP_STAGE_RHS( xr, xth, xpr, xpth)
        }
        GP_HENON(dp.B5)
        ar = o.dr; ath = o.dth; apr = o.dpr; apth = o.dpth;                         // K5
        sts2(KS(6), ar, ath); sts2(KS(7), apr, apth);
        bt += dp.B5 * o.dt; bph += dp.B5 * o.dph;
        qet += dp.E5 * o.dt; qeph += dp.E5 * o.dph;
        // stage 6
        {
          double xr = fma(dp.A65, ar, fma(dp.A61, hk1r, r)), xth = fma(dp.A65, ath, fma(dp.A61, hk1th, thb));
          double xpr = fma(dp.A65, apr, fma(dp.A61, hk1pr, pr)), xpth = fma(dp.A65, apth, fma(dp.A61, hk1pth, pth));
          lds2(KS(0), br, bth); lds2(KS(1), bpr, bpth);                             // K2
          xr = fma(dp.A62, br, xr); xth = fma(dp.A62, bth, xth); xpr = fma(dp.A62, bpr, xpr); xpth = fma(dp.A62, bpth, xpth);
          lds2(KS(2), br, bth); lds2(KS(3), bpr, bpth);                             // K3
          xr = fma(dp.A63, br, xr); xth = fma(dp.A63, bth, xth); xpr = fma(dp.A63, bpr, xpr); xpth = fma(dp.A63, bpth, xpth);
          lds2(KS(4), br, bth); lds2(KS(5), bpr, bpth);                             // K4
          xr = fma(dp.A64, br, xr); xth = fma(dp.A64, bth, xth); xpr = fma(dp.A64, bpr, xpr); xpth = fma(dp.A64, bpth, xpth);
          GP_STAGE_RHS( xr, xth, xpr, xpth)
        }
        GP_HENON(dp.B6)
        ar = o.dr; ath = o.dth; apr = o.dpr; apth = o.dpth;                         // K6
        bt += dp.B6 * o.dt; bph += dp.B6 * o.dph;
        qet += dp.E6 * o.dt; qeph += dp.E6 * o.dph;
#undef GP_HENON
        // trial end state (5th-order solution; a7 = b) and the error sums without e7 k7
        {
          double xr = fma(dp.B6, ar, fma(dp.B1, hk1r, r)), xth = fma(dp.B6, ath, fma(dp.B1, hk1th, th));
          double xpr = fma(dp.B6, apr, fma(dp.B1, hk1pr, pr)), xpth = fma(dp.B6, apth, fma(dp.B1, hk1pth, pth));
          er = dp.E1 * hk1r + dp.E6 * ar; eth = dp.E1 * hk1th + dp.E6 * ath;
          epr = dp.E1 * hk1pr + dp.E6 * apr; epth = dp.E1 * hk1pth + dp.E6 * apth;
          lds2(KS(2), br, bth); lds2(KS(3), bpr, bpth);                             // K3
          xr = fma(dp.B3, br, xr); xth = fma(dp.B3, bth, xth); xpr = fma(dp.B3, bpr, xpr); xpth = fma(dp.B3, bpth, xpth);
          er += dp.E3 * br; eth += dp.E3 * bth; epr += dp.E3 * bpr; epth += dp.E3 * bpth;
          lds2(KS(4), br, bth); lds2(KS(5), bpr, bpth);                             // K4
          xr = fma(dp.B4, br, xr); xth = fma(dp.B4, bth, xth); xpr = fma(dp.B4, bpr, xpr); xpth = fma(dp.B4, bpth, xpth);
          er += dp.E4 * br; eth += dp.E4 * bth; epr += dp.E4 * bpr; epth += dp.E4 * bpth;
          lds2(KS(6), br, bth); lds2(KS(7), bpr, bpth);                             // K5
          xr = fma(dp.B5, br, xr); xth = fma(dp.B5, bth, xth); xpr = fma(dp.B5, bpr, xpr); xpth = fma(dp.B5, bpth, xpth);
          er += dp.E5 * br; eth += dp.E5 * bth; epr += dp.E5 * bpr; epth += dp.E5 * bpth;
          nr = xr; nth = xth; npr = xpr; npth = xpth;
        }
        nt = lds1(CS(C_T)) + bt;
        nph = lds1(CS(C_PH)) + bph;
        nlam = lds1(CS(C_LAM)) + s * bl;
        et = qet;
        eph = qeph;
#undef GP_STAGE_RHS
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
