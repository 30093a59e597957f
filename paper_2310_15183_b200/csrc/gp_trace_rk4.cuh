// gp_trace_rk4.cuh — persistent classical RK4 kernel (schemes 0 and 1; PAPER.md L257-278,
// eq 42-49 with reading R9; step h fixed, or h_n = h_rel r_n per reading R17).
// Included by gp_trace.cuh.
//
// Every trip of the loop is one RK4 step per lane: an ordinary step, or a landing step of the
// same formula on dy/ds = F/F_w (reading R14).  Reading R31: in an ordinary step each state the
// equations are evaluated at is first tested against the capture radius; the first hit ends the
// ray as CAPTURED (then one landing step from y_n).
//
// T is the arithmetic type of Hamilton's equations and S that of the state and of the Runge-Kutta sums:
// (double, double) is the required path; (float, float) the single-precision variant BASELINE.json
// configs[4] asks for (cfg.precision = 1); (float, double) the mixed variant of SURVEY.md section 8(f)
// NEXT-1 (cfg.precision = 2): the equations are evaluated in FP32 at the state rounded to FP32, their
// results are accumulated into an FP64 state, so that rounding no longer accumulates with the number of
// steps.  The ray is always born in double (rows a2, a3) and the record is always written in double.
#ifndef GP_TRACE_RK4_CUH_
#define GP_TRACE_RK4_CUH_

namespace gp {
#if defined(__CUDACC__)

constexpr int kParkSlotsRk4 = 7;  // trial state (r, th, pr, pth, t, ph, lambda) across an equator landing
constexpr int kBirthQueueDoubles = 9;   // per queued ray (see the kernel)
constexpr int kBirthQueueStride = kBirthQueueDoubles * 32 + 2;   // + the slot of entry 0 (and a pad), per warp
constexpr size_t kBirthQueueBytes = (size_t)(kBlock / 32) * kBirthQueueStride * sizeof(double);

// Rows a2 + a3 and the reference value of the Carter monitor for one queued ray; e[k * 32], k = 0..8.
// Out of line on purpose: it runs once per 32 rays with every lane's ray state live around it, and inlined its
// FP64 temporaries came on top of that state (158 registers instead of 122 in the FP64 kernel); as a call it
// costs a few saves and restores around a cold path.
template <int METRIC>
__device__ __noinline__ void birth_to_queue(const CameraConst &cc, const MetricConst &mc, long long ray, double *e) {
  double dr0, dth0, dph0, dpt, dpr, dpth, dpph, q0 = 0.0, iq0 = 1.0;
  ray_birth(cc, mc, ray, dr0, dth0, dph0, dpt, dpr, dpth, dpph);
  if (METRIC != METRIC_MN) {
    // Reference value of the Carter monitor (R23), once per ray, from the initial state (H = 0 there by
    // construction, so the term in H is left out: a 1e-16 relative difference to the value taken at the
    // first step) — the per-step monitor then carries no "first step" instructions.
    double s0, c0;
    sincos(dth0, &s0, &c0);
    const double a2 = (METRIC == METRIC_KERR) ? mc.a2 : 0.0;
    q0 = dpth * dpth + c0 * c0 * (dpph * dpph / (s0 * s0) - a2 * dpt * dpt);
    iq0 = 1.0 / fmax(1.0, fabs(q0));
  }
  e[0 * 32] = dr0; e[1 * 32] = dth0; e[2 * 32] = dph0; e[3 * 32] = dpt; e[4 * 32] = dpr;
  e[5 * 32] = dpth; e[6 * 32] = dpph; e[7 * 32] = q0; e[8 * 32] = iq0;
}

template <bool B> struct LandTag { static constexpr bool value = B; };

// Resident blocks per SM asked of ptxas (0 = its own choice), by variant:
//   FP64 Manko-Novikov                        2  (the duals need up to 255 registers)
//   Manko-Novikov with FP32 equations         4 without an object (128 registers), 3 with one (168; at 128 one
//                                                of them spills a word)
//   FP64 Schwarzschild / Kerr                 4  (128 registers; the out-of-line batch birth is saved around.  With
//                                                an object too since the step was split and the birth moved out of
//                                                line: Kerr + disk at 1024^2 15.00 -> 14.05 ms, + ring 11.52 -> 10.91)
//   FP32 state, no object, Schw. / Kerr       5  (96 registers; measured on B200 at 4096^2: 137.2 ms with four
//                                                blocks, 129.8 with five, 130.2 with six, 131.3 with eight)
//   FP32 with an object, FP32 equations + FP64 state (Schwarzschild / Kerr)   4
template <int METRIC, int OBJ, class T, class S>
constexpr int rk4_min_blocks() {
  if (METRIC == METRIC_MN) return sizeof(T) == 8 ? 2 : (OBJ == 0 ? 4 : 3);
  if (sizeof(T) == 8) return 4;
  return (sizeof(S) == 4 && OBJ == 0) ? 5 : 4;
}

// OBJ: 0 no object; 1 thin disk, crossings located and recorded (R19); 2 solid ring, the ray ends where it
// enters the volume (R39).  Both objects use the park area.
template <int METRIC, int OBJ, class T, class S = T>
__global__ void __launch_bounds__(kBlock, rk4_min_blocks<METRIC, OBJ, T, S>()) trace_rk4(const __grid_constant__ TraceParams P) {
  constexpr bool DISK = (OBJ == 1), RING = (OBJ == 2);
  extern __shared__ double park_raw[];  // [kParkSlotsRk4][kBlock] of S when OBJ != 0
  S *park = reinterpret_cast<S *>(park_raw);
  const MetricConst &mc = P.mc;
  const int tid = threadIdx.x;
  const S r_cap = (S)P.r_cap, r_esc = (S)P.r_esc, half_pi = (S)kHalfPi;
  // per-launch constants in the state's type: for S = float they are read from the parameter block as FP32
  // operands (converted once on the host) instead of being converted from double in every step
  constexpr bool kF32 = (sizeof(S) == 4);
  const S h_fix = kF32 ? (S)P.h_f : (S)P.h, h_rel = kF32 ? (S)P.h_rel_f : (S)P.h_rel;
  const S lam_max = kF32 ? (S)P.lambda_max_f : (S)P.lambda_max;   // lambda_max_f: smallest float >= lambda_max
  const S sixth = kF32 ? S(1.0 / 6.0) : (S)dp.sixth;

  int mode = MODE_IDLE;
  long long slot = -1;
  T pt = T(0), pph = T(0);
  S t = S(0), r = S(0), th = S(0), ph = S(0), pr = S(0), pth = S(0), lam = S(0);
  S target = S(0);
  // (err_margin belongs to the adaptive scheme: +inf in every fixed-step record, a constant that needs no register)
  MonitorsT<T> mo = {T(0), T(0), T(0), T(1), T(0), (T)__longlong_as_double(0x7ff0000000000000LL)};
  unsigned n_acc = 0, n_cross = 0, n_rec = 0, n_land = 0, status = 0;
  unsigned tot_rays = 0, tot_steps = 0, tot_rhs = 0;   // per lane: < 2^32 (rays per lane x the step budget x 4)
// the ray goes on from the trial state parked before a landing step (thin disk: always; ring: no hit); the
// ring variant counts the equator crossing of that step here, as the oracle does after its ring test
#define GP_RESUME_PARKED()                                                                    \
  {                                                                                           \
    const S *pk = park + tid;                                                                 \
    if (RING && (th - half_pi) * (pk[1 * kBlock] - half_pi) < S(0)) ++n_cross;                \
    r = pk[0 * kBlock]; th = pk[1 * kBlock]; pr = pk[2 * kBlock]; pth = pk[3 * kBlock];       \
    t = pk[4 * kBlock]; ph = pk[5 * kBlock]; lam = pk[6 * kBlock];                            \
    mode = MODE_NORMAL;                                                                       \
  }
  // Birth queue: rays are fetched and born (rows a1-a3) 32 at a time by the whole warp and handed to lanes as
  // they fall idle.  A lane that refilled alone ran the birth — 400 instructions, a quarter of them FP64 — for
  // the whole warp with 31 lanes masked off: 7 % of the FP32 kernel's issue slots.  Near the end of the image
  // (fewer than two rays per lane left) a warp fetches only what it needs, so that no ray waits in one warp's
  // queue while another warp idles; the Manko-Novikov kernels, whose ray lengths differ by a factor of 700,
  // always do.  Entry: r, theta, phi, p_t, p_r, p_theta, p_phi, Q0, 1/max(1,|Q0|).
  constexpr int kQ = kBirthQueueDoubles;
  const unsigned lane = (unsigned)tid & 31u;
  double *bq = park_raw + (OBJ != 0 ? (sizeof(S) * kBlock * kParkSlotsRk4) / 8 : 0) + (tid >> 5) * kBirthQueueStride;
  long long *q_base_p = reinterpret_cast<long long *>(bq + kQ * 32);   // slot of entry 0 (read when a lane refills)
  if (lane == 0u) *q_base_p = 0;
  __syncwarp();
  int q_n = 0, q_head = 0;      // warp-uniform: entries in the queue, entries handed out
  bool drained = false;         // the work counter has passed the end of the image
  bool none_left = false;       // ... and the queue is empty: idle lanes stay idle (warp-uniform)
  stamp_start(P.counters);

  for (;;) {
    // ---- a1: refill idle lanes, from the warp's birth queue ----
    const bool need = (mode == MODE_IDLE) && !none_left;
    const unsigned need_mask = __ballot_sync(kFull, need);
    if (need_mask) {
      if (q_head == q_n && !drained) {
        // a1 + a2 + a3 for a batch: one atomic for the warp, the rays born by all lanes at once
        // Manko-Novikov: always exact.  Its shadow rays run to the step budget, 700 x a normal ray, and come
        // in runs of neighbouring pixels: a batch of them would wait in one warp's queue for that warp's own
        // lanes, each busy for a second (measured, config 5b at 512^2: 1.90 s with batches, 1.12 s without).
        const bool tail = METRIC == METRIC_MN ||
                          *q_base_p + q_n >= P.cc.ray_count - 2LL * (long long)gridDim.x * kBlock;
        const int want = tail ? __popc(need_mask) : 32;
        unsigned long long base = 0;
        if (lane == 0u) base = atomicAdd(P.counters, (unsigned long long)want);
        base = __shfl_sync(kFull, base, 0);
        const long long left = P.cc.ray_count - (long long)base;
        const long long q_base = (long long)base;
        if (lane == 0u) *q_base_p = q_base;
        q_n = left >= (long long)want ? want : (left > 0 ? (int)left : 0);
        q_head = 0;
        drained = left <= (long long)want;   // the counter is past the image: nothing more will come
        if ((int)lane < q_n) birth_to_queue<METRIC>(P.cc, mc, P.cc.ray_begin + (q_base + lane) * P.cc.ray_stride, bq + lane);
        __syncwarp();
      }
      const int avail = q_n - q_head;
      if (need) {
        const int rank = __popc(need_mask & ((1u << lane) - 1u));
        if (rank < avail) {
          const double *e = bq + (q_head + rank);
          slot = *q_base_p + (q_head + rank);
          r = (S)e[0 * 32]; th = (S)e[1 * 32]; ph = (S)e[2 * 32]; pt = (T)e[3 * 32]; pr = (S)e[4 * 32];
          pth = (S)e[5 * 32]; pph = (T)e[6 * 32];
          mo.Q0 = (T)e[7 * 32]; mo.iQ0 = (T)e[8 * 32];
          t = S(0); lam = S(0);
          mode = MODE_NORMAL;
          n_acc = n_cross = n_rec = n_land = 0;
          mo.h_max = T(0); mo.q_drift = T(0);
          mo.sin_min = (T)__longlong_as_double(0x7ff0000000000000LL);
        }   // else: the queue ran out under this lane; it is refilled in the next trip (if anything is left)
      }
      const int asked = __popc(need_mask);
      q_head += asked < avail ? asked : avail;
      none_left = drained && q_head == q_n;
      __syncwarp();
    }
    if (!__any_sync(kFull, mode != MODE_IDLE)) break;

    if (mode != MODE_IDLE) {
      bool finished = false;
      // stop tests at the top of every ordinary step (R18)
      if (mode == MODE_NORMAL && (n_acc >= (unsigned)P.max_steps || lam >= lam_max)) {
        status = GP_RAY_MAXSTEPS;
        finished = true;
      }
      // Landing steps are 1 in several hundred per lane.  The step is compiled twice: LAND = false is the
      // ordinary step and nothing else (no Henon divisor, no mode selects, no landing bookkeeping) and runs
      // whenever no lane of this convergence group is landing — nine warp-steps in ten; LAND = true is the
      // same instruction stream with the per-lane reciprocal selector (gp_trace.cuh, reading R14).
      bool any_land = false;   // some lane of this convergence group is landing (set before the call)
      auto step = [&](auto land_tag) {
        constexpr bool LAND = decltype(land_tag)::value;
        const bool normal = LAND ? (mode == MODE_NORMAL) : true;
        const bool land_r = LAND ? (mode == MODE_LAND_R) : false;
        const S s = normal ? (P.scheme == 0 ? h_fix : h_rel * r) : (land_r ? (target - r) : (target - th));
        S sl = S(1);  // weighted sum of 1/F_w: d(lambda)/ds of a landing step (unused otherwise)
#define GP_HENON(weight, first)                                                   \
  if (LAND && any_land) {                                                         \
    T iv = normal ? T(1) : frcp(land_r ? o.dr : o.dth);                           \
    o.dt *= iv; o.dr *= iv; o.dth *= iv; o.dph *= iv; o.dpr *= iv; o.dpth *= iv;  \
    sl = (first) ? (S)iv : sl + S(weight) * (S)iv;                                \
  }
        RhsT<T> o;
        // k1 = F(y_n)
        rhs_eval<METRIC>(mc, pt, pph, (T)r, (T)th, (T)pr, (T)pth, o);
        if (normal)
          monitor_apply<METRIC>(mo, (T)fabs(T(0.5) * o.H2), carter_q<METRIC>(mc, pt, pph, (T)pth, o), (T)fabs(o.s),
                                false);
        GP_HENON(1.0, true)
        // Stage angles (Schwarzschild, Kerr): sin, cos of theta_n + d from (sin, cos) theta_n — by-products of
        // k1 — through the addition theorems: no range reduction or quadrant logic in stages 2-4.  A fixed
        // step has no error control to reject a stage that swings theta by more than the Taylor kernels
        // cover (a ray grazing the polar axis does), so |d| > 1/4 takes the full evaluation.
        constexpr bool kAngle = (METRIC != METRIC_MN);
        const T sn_ = o.s, cn_ = o.c;
#define GP_STAGE(yr_, dth_, ypr_, ypth_)                                                          \
  if (kAngle && fabs((T)(dth_)) <= T(0.25)) {                                                     \
    T ss_, cc_;                                                                                   \
    sincos_add(sn_, cn_, (T)(dth_), &ss_, &cc_);                                                  \
    rhs_eval_sc<METRIC>(mc, pt, pph, (T)(yr_), ss_, cc_, (T)(ypr_), (T)(ypth_), o);               \
  } else {                                                                                        \
    rhs_eval<METRIC>(mc, pt, pph, (T)(yr_), (T)(th + (dth_)), (T)(ypr_), (T)(ypth_), o);          \
  }
        // k1 + 2k2 + 2k3 + k4, accumulated in the state's type
        S st = (S)o.dt, sr = (S)o.dr, sth = (S)o.dth, sph = (S)o.dph, spr = (S)o.dpr, spth = (S)o.dpth;
        const S hs = S(0.5) * s;
        // k2 = F(y_n + h/2 k1)
        S yr = r + hs * (S)o.dr;
        bool captured = normal && (yr < r_cap);
        GP_STAGE(yr, hs * (S)o.dth, pr + hs * (S)o.dpr, pth + hs * (S)o.dpth)
        GP_HENON(2.0, false)
        st += S(2) * (S)o.dt; sr += S(2) * (S)o.dr; sth += S(2) * (S)o.dth; sph += S(2) * (S)o.dph;
        spr += S(2) * (S)o.dpr; spth += S(2) * (S)o.dpth;
        // k3 = F(y_n + h/2 k2)
        yr = r + hs * (S)o.dr;
        captured = captured || (normal && (yr < r_cap));
        GP_STAGE(yr, hs * (S)o.dth, pr + hs * (S)o.dpr, pth + hs * (S)o.dpth)
        GP_HENON(2.0, false)
        st += S(2) * (S)o.dt; sr += S(2) * (S)o.dr; sth += S(2) * (S)o.dth; sph += S(2) * (S)o.dph;
        spr += S(2) * (S)o.dpr; spth += S(2) * (S)o.dpth;
        // k4 = F(y_n + h k3)
        yr = r + s * (S)o.dr;
        captured = captured || (normal && (yr < r_cap));
        GP_STAGE(yr, s * (S)o.dth, pr + s * (S)o.dpr, pth + s * (S)o.dpth)
        GP_HENON(1.0, false)
        st += (S)o.dt; sr += (S)o.dr; sth += (S)o.dth; sph += (S)o.dph; spr += (S)o.dpr; spth += (S)o.dpth;
#undef GP_HENON
#undef GP_STAGE
        const S w = s * sixth;
        const S nt = t + w * st, nr = r + w * sr, nth = th + w * sth, nph = ph + w * sph,
                npr = pr + w * spr, npth = pth + w * spth;

        if (normal) {
          const S ysum = ((nt + nr) + (nth + nph)) + (npr + npth);
          const bool nonfinite = !captured && !finite_d(ysum);
          if (!nonfinite) ++n_acc;
          if (nonfinite) {
            status = GP_RAY_NONFINITE;   // record = last finite state y_n
            finished = true;
          } else if (captured || nr > r_esc || nr < r_cap) {
            const bool esc = !captured && nr > r_esc;
            status = esc ? GP_RAY_ESCAPED : GP_RAY_CAPTURED;
            target = esc ? r_esc : r_cap;
            mode = MODE_LAND_R;
          } else {
            bool commit = true;
#define GP_PARK()                                                                                      \
  {                                                                                                    \
    S *pk = park + tid;                                                                                \
    pk[0 * kBlock] = nr; pk[1 * kBlock] = nth; pk[2 * kBlock] = npr; pk[3 * kBlock] = npth;            \
    pk[4 * kBlock] = nt; pk[5 * kBlock] = nph; pk[6 * kBlock] = lam + s;                               \
  }
            bool ring_try = false;
            if (RING) {
              // R39: the step can meet the box r_in..r_out x |theta - pi/2| <= d only if every coordinate that
              // starts outside its interval ends inside it or beyond it (see gp_trace_dp54.cuh, gp.h)
              const S rin = (S)P.disk_r_in, rout = (S)P.disk_r_out, rd = (S)P.ring_d;
              const S un = th - half_pi, un1 = nth - half_pi;
              const bool th_out = fabs(un) > rd;
              const bool r_out_n = !(r >= rin && r <= rout);
              const bool th_enters = fabs(un1) <= rd || un * un1 < S(0);
              const bool r_enters = (nr >= rin && nr <= rout) || ((r < rin) != (nr < rin));
              ring_try = (th_out || r_out_n) && (!th_out || th_enters) && (!r_out_n || r_enters);
              if (ring_try) {
                GP_PARK()
                if (th_out) {
                  target = half_pi + (un > S(0) ? rd : -rd);
                  mode = MODE_LAND_TH;
                } else {
                  status = GP_RAY_HIT_RING;
                  target = (r < rin) ? rin : rout;
                  mode = MODE_LAND_R;
                }
                commit = false;
              }
            }
            if (!ring_try && (th - half_pi) * (nth - half_pi) < S(0)) {
              ++n_cross;
              if (DISK && n_rec < (unsigned)P.max_crossings) {
                GP_PARK()
                target = half_pi;
                mode = MODE_LAND_TH;
                commit = false;
              }
            }
#undef GP_PARK
            if (commit) {
              t = nt; r = nr; th = nth; ph = nph; pr = npr; pth = npth; lam += s;
            }
          }
        } else if (land_r) {
          ++n_land;
          bool resume = false;
          if (RING && status == GP_RAY_HIT_RING) {
            // radial face of the ring: a hit if the landed theta is inside the slab, else the ray goes on
            if (fabs(nth - half_pi) <= (S)P.ring_d) {
              P.disk[slot].r_cross[0] = (double)target;
              P.disk[slot].g[0] = kepler_g<METRIC>(mc, (double)target, (double)pt, (double)pph);
              n_rec = 1;
            } else {
              status = 0;
              resume = true;
            }
          }
          if (!resume) {
            t = nt; r = target; th = nth; ph = nph; pr = npr; pth = npth; lam = lam + w * sl;
            finished = true;
          } else {
            GP_RESUME_PARKED()
          }
        } else {  // MODE_LAND_TH
          ++n_land;
          if (RING) {
            const S rin = (S)P.disk_r_in, rout = (S)P.disk_r_out;
            if (nr >= rin && nr <= rout) {          // theta-face hit: the record is the landed state
              P.disk[slot].r_cross[0] = (double)nr;
              P.disk[slot].g[0] = kepler_g<METRIC>(mc, (double)nr, (double)pt, (double)pph);
              n_rec = 1;
              status = GP_RAY_HIT_RING;
              t = nt; r = nr; th = target; ph = nph; pr = npr; pth = npth; lam = lam + w * sl;
              finished = true;
            } else if (!(r >= rin && r <= rout)) {  // try the radial face on y_n's side
              status = GP_RAY_HIT_RING;
              target = (r < rin) ? rin : rout;
              mode = MODE_LAND_R;
            } else {
              GP_RESUME_PARKED()
            }
          }
          if (DISK) {
            const double rc = (double)nr;
            if (rc >= P.disk_r_in && rc <= P.disk_r_out) {
              P.disk[slot].r_cross[n_rec] = rc;
              P.disk[slot].g[n_rec] = kepler_g<METRIC>(mc, rc, (double)pt, (double)pph);
              ++n_rec;
            }
            GP_RESUME_PARKED()
          }
          if (OBJ == 0) mode = MODE_NORMAL;
        }
      };
      if (!finished) {
        // (Manko-Novikov: one copy, with the divisor work behind the warp-uniform flag; the rest of the landing
        // logic is nothing beside its dual-number evaluations)
        any_land = __any_sync(__activemask(), mode != MODE_NORMAL);
        if (METRIC == METRIC_MN || any_land) step(LandTag<true>());
        else step(LandTag<false>());
      }

      if (finished) {
        const unsigned n_rhs = 4u * n_acc + 3u * n_land;
        Monitors mod = {(double)mo.h_max, (double)mo.q_drift, 0.0, 0.0, (double)mo.sin_min, (double)mo.err_margin};
        // the exit surface is exact in the record whatever the arithmetic type
        // (a ring hit on a radial face has r = that face, exact in S already)
        const double r_rec = (status == GP_RAY_ESCAPED) ? P.r_esc : (status == GP_RAY_CAPTURED ? P.r_cap : (double)r);
        store_record(P.rays + slot, (double)t, r_rec, (double)th, (double)ph, (double)pr, (double)pth, (double)lam,
                     (double)pt, (double)pph, mod, status, n_acc, 0u, n_cross, n_rec, n_rhs);
        if (OBJ != 0) {
          const double qnan = __longlong_as_double(0x7ff8000000000000LL);
          for (unsigned i = n_rec; i < 3u; ++i) {
            P.disk[slot].r_cross[i] = qnan;
            P.disk[slot].g[i] = qnan;
          }
        }
        stamp_ray_done(P.counters, P.cc.ray_count);
        tot_rays += 1; tot_steps += n_acc; tot_rhs += n_rhs;
        mode = MODE_IDLE;
      }
    }
  }

  if (tot_rays) {
    atomicAdd(P.counters + 1, (unsigned long long)tot_rays);
    atomicAdd(P.counters + 2, (unsigned long long)tot_steps);
    atomicAdd(P.counters + 3, (unsigned long long)tot_rhs);
  }
  stamp_end(P.counters);
}

#endif  // __CUDACC__
}  // namespace gp
#endif
