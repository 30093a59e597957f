/* gp.h — C-ABI of the B200-native null-geodesic tracer (libgp.so).
 *
 * The library integrates one null geodesic per image pixel through a stationary,
 * axisymmetric spacetime in Hamiltonian form,
 *     H(q,p) = 1/2 g^{mu nu}(q) p_mu p_nu = 0                      (eq 3)
 *     dq^mu/dlambda = g^{mu nu} p_nu                                (eq 4 / L678, eq 102)
 *     dp_mu/dlambda = -1/2 (d_mu g^{rho sigma}) p_rho p_sigma       (eq 103; eq 5 at L122 lacks the 1/2)
 * with explicit Runge-Kutta steps (eq 42-49), from a camera until the
 * ray is captured or leaves a bounding sphere (section 3.3.2; L404, section 5.1).
 * Every step of the path runs in hand-written CUDA kernels for sm_100a; there is no CPU
 * fallback.  All device buffers are owned by the caller; the library allocates nothing
 * persistent and never synchronises the device (except gp_trace_host, which says so).
 *
 * Conventions: G = c = 1; coordinates (t, r, theta, phi) are Schwarzschild /
 * Boyer-Lindquist (eq 8, L147-159 eq 9-14, L181-230 eq 20-39);
 * DESIGN.md section 3 lists every reading taken where the paper is silent or garbled.
 */
#ifndef GP_H_
#define GP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GP_VERSION 103 /* major*10000 + minor*100 + patch */
/* Capacity of the library's static scratch, in rays (one 1024 x 1024 image): gp_trace_static only. */
#define GP_STATIC_MAX_RAYS 1048576

/* ---- spacetimes (section 2.2) ------------------------------------------- */
enum {
  GP_SCHWARZSCHILD = 0, /* PAPER.md L136, eq 8                                          */
  GP_KERR = 1,          /* PAPER.md L147-159, eq 9-14, Boyer-Lindquist                  */
  GP_MANKO_NOVIKOV = 2  /* PAPER.md L181-230, eq 20-39, quadrupole deviation only       */
};

/* M: mass; a = S/M: spin length (eq 14); q: Manko-Novikov quadrupole deviation (eq 25,
 * beta = q M^3 / k^3).  Schwarzschild ignores a and q; Kerr ignores q.
 * Valid: M > 0 (M = 0 allowed for GP_SCHWARZSCHILD only: flat space, capture test off);
 * |a| < M; GP_MANKO_NOVIKOV needs a != 0 (eq 23 divides by S/M). */
typedef struct gp_metric_params {
  double M, a, q;
} gp_metric_params;

/* ---- camera: pinhole at (r_obs, theta_obs, phi_obs), ZAMO orthonormal tetrad --------
 * Replaces PAPER.md L314-348 (section 3.3.1) per BASELINE.json; see DESIGN.md section 3.
 * Ray index -> pixel: with S = supersample, Wt = width*S, Ht = height*S,
 *   ray -> (I, J) = (ray mod Wt, ray div Wt);  J = 0 is the beta_min row.
 *   X = (I + 0.5)/S + jit_x + shift_x_px,  Y = (J + 0.5)/S + jit_y + shift_y_px   [pixels]
 *   alpha = alpha_min + X*((alpha_max-alpha_min)/width),  beta likewise with height.
 * jit = (2u-1)*jitter_amp_px, u from a SplitMix64 hash of (jitter_seed, ray, axis);
 * the map is evaluated with individually rounded operations and is bit-exact against the
 * oracle.  Rays traced by a call: ray_begin + k*ray_stride for k in [0, ray_count);
 * record k is written at slot k of the output buffers.                                 */
typedef struct gp_camera {
  double r_obs, theta_obs, phi_obs;
  double alpha_min, alpha_max, beta_min, beta_max; /* image-plane window, units of length */
  int32_t width, height;                           /* pixels, > 0                         */
  int32_t supersample;                             /* S >= 1: S x S sub-rays per pixel    */
  int32_t projection;                              /* 0 = pinhole in the ZAMO tetrad; 1 = the paper's
                                                      Euclidean screen (below)             */
  uint64_t jitter_seed;
  double jitter_amp_px;          /* 0 = sub-pixel centres; 0.5 = uniform in +-0.5 px      */
  double shift_x_px, shift_y_px; /* rigid shift of the whole grid (chaos companion run)   */
  int64_t ray_begin, ray_count, ray_stride; /* ray_stride >= 1; all rays < Wt*Ht          */
  /* projection = 1, PAPER.md L314-348 (section 3.3.1, Fig 2-3, eq 51-55): a flat screen in the
   * Euclidean xyz of eq 51-53, centred at r_obs c_hat (c_hat = unit vector at theta_obs, phi_obs),
   * spanned by e_phi (alpha) and e_up = -e_theta (beta).  Pixel (alpha, beta) starts AT
   * r_obs c_hat + alpha e_phi + beta e_up with direction -c_hat + focal_2f_over_d (alpha e_phi +
   * beta e_up) (0 = parallel rays, "focal distance infinity"); position and direction go to
   * Boyer-Lindquist by inverting eq 51-53 (a = the metric's spin), dt/dlambda solves eq 54 and the
   * ray is scaled to dt/dlambda = -1 before eq 55 lowers the index.  Needs r_escape beyond every
   * start point.  Ignored when projection = 0.                                                  */
  double focal_2f_over_d;
} gp_camera;

/* ---- integrator ---------------------------------------------------------------------
 * scheme 0: classical RK4, fixed step h                     (eq 42-49)
 * scheme 1: classical RK4, h_n = h_rel * r_n                (BASELINE.json configs[4])
 * scheme 2: Dormand-Prince 5(4) embedded pair, FSAL, max-norm error over the six evolving
 *           components, sc = atol + rtol*max(|y|,|y+|), fac = 0.9*err^(-1/5) clamped to
 *           [0.2, 5], cap h <= h_cap_rel * r, h0 = h_cap_rel * r_obs
 *           (BASELINE.json configs[1-3], reading R10).
 * A ray ends: ESCAPED when a step lands at r > r_escape, CAPTURED when it lands at
 * r < r_H*(1+eps_capture) (both followed by one landing step onto that surface with r as
 * the independent variable), MAXSTEPS after max_steps attempted steps (or lambda >=
 * lambda_max when lambda_max > 0), NONFINITE / STEP_UNDERFLOW on numerical failure.     */
typedef struct gp_integrator_cfg {
  int32_t scheme;    /* 0, 1, 2 as above                                                 */
  int32_t precision; /* 0 = FP64 (required path).
                        1 = FP32 state and equations, schemes 0 and 1 only (scheme 2 -> GP_E_UNSUPPORTED).
                        2 = mixed: Hamilton's equations in FP32 at the state
                            rounded to FP32, state / Runge-Kutta sums / error norm / controller in FP64;
                            all schemes; with scheme 2 rtol and atol must be >= 1e-7 (the error estimate
                            carries the 6e-8 noise of an FP32 evaluation; below -> GP_E_BAD_PARAM).
                            Stated tolerance of 1 and 2: DESIGN.md 7.6.
                        The ray is born and the record written in FP64 in every case; other values ->
                        GP_E_UNSUPPORTED                                                             */
  double h, h_rel, rtol, atol, h_cap_rel;
  int64_t max_steps; /* attempted steps (accepted + rejected), landing steps not counted */
  double lambda_max; /* <= 0: off                                                        */
  double eps_capture, r_escape;
  double disk_r_in, disk_r_out; /* thin equatorial disk; disk_r_in <= 0 -> prograde ISCO  */
  int32_t max_crossings;        /* 0..3 recorded disk crossings; 0 = disk off             */
  int32_t segment_steps;        /* Manko-Novikov with scheme 2 only (ignored otherwise): rays that stall near the
                                   singular horizon run to max_steps, hundreds of
                                   times a normal ray.  After this many attempted steps a ray's state is parked
                                   in its own record and redistributed over all lanes by a further launch of
                                   the same kernel on the same stream; results are identical
                                   bit for bit, only the balance changes.  0 = off (the default: measured gain
                                   0.5 % on config 4, 4 % at 1024^2), -1 = the library's choice of segment
                                   (max(4096, max_steps / 48)), > 0 = that many steps (at most 4096 rounds,
                                   else GP_E_BAD_PARAM; < -1 -> GP_E_BAD_PARAM).  While such a call is in flight it holds
                                   16 bytes of stream-ordered scratch per ray from the library's pool.      */
  /* > 0: a SOLID RING instead of the thin disk (objects "cannot be infinitely thin, as
   * their collision is based on the ray propagating to a point inside volume of the object"; L735-743,
   * Figs 15-17: "a region in space around the equator" whose hits go "through the redshift
   * calculation").  Volume: disk_r_in <= r <= disk_r_out, |theta - pi/2| <= ring_half_angle (a box in
   * r, theta).  Opaque: the ray ends with status GP_RAY_HIT_RING at the point where it ENTERS the
   * volume.  An accepted, non-terminal step y_n -> y_{n+1} is examined when every coordinate (r, theta)
   * that starts outside its interval ends inside it or beyond it; the entry is located from y_n by the
   * landing step (R14) on the theta-face on y_n's side (a hit if the landed radius is in range),
   * else on the radial face on y_n's side (a hit if the landed theta is in the slab); otherwise the ray
   * goes on from y_{n+1} (reading R39).  The record holds the state at the hit; disk record
   * slot 0 holds the hit radius and g of the circular equatorial emitter at that radius (eq 56-57), the
   * other slots NaN.  Every scheme and precision (the landing steps use the scheme's own formula).  Requires max_crossings = 0 and a disk buffer; Manko-Novikov needs an explicit
   * disk_r_in.  0 = no ring.  Values < 0 or >= 1.5 -> GP_E_BAD_PARAM; with max_crossings > 0 ->
   * GP_E_UNSUPPORTED.                                                              */
  double ring_half_angle;
} gp_integrator_cfg;

/* ---- outputs ------------------------------------------------------------------------ */
enum {
  GP_RAY_ESCAPED = 0,
  GP_RAY_CAPTURED = 1,
  GP_RAY_MAXSTEPS = 2,
  GP_RAY_NONFINITE = 3,
  GP_RAY_STEP_UNDERFLOW = 4,
  GP_RAY_HIT_RING = 5 /* ended on the solid ring (cfg.ring_half_angle > 0) */
};

/* One per ray, 128 bytes.  theta and phi are raw (accumulated, not wrapped).  The traced
 * covector is the time-reversed one: p_t > 0 is the photon energy measured at infinity per
 * unit locally (ZAMO) measured energy, and L_z = -p_phi (reading R12).        */
typedef struct gp_ray_record {
  /* bytes 0-31 */
  double t, r, theta, phi; /* state on the exit surface (or last state)                   */
  /* bytes 32-63: with the sector above, everything image formation reads (gp_shade)     */
  double lambda;           /* affine parameter at exit                                     */
  uint32_t status;         /* GP_RAY_*                                                     */
  uint32_t n_accepted;
  double p_r, p_theta;     /* rest of the exit state                                       */
  /* bytes 64-95 */
  double p_t, p_phi;       /* constants of the ray                                         */
  double h_max;            /* max |H| over every state a step was attempted from          */
  double q_drift;          /* Kerr/Schwarzschild: max |Q-Q0| / max(1,|Q0|), Carter constant */
  /* bytes 96-127 */
  double sin_theta_min;    /* min |sin theta| over the same states                         */
  double err_margin;       /* scheme 2: min |err-1| over attempted steps; else +inf        */
  uint32_t n_rejected;
  uint32_t n_equator_crossings; /* sign changes of theta - pi/2 over accepted steps       */
  uint32_t n_disk_recorded;     /* crossings with disk_r_in <= r <= disk_r_out, <= 3      */
  uint32_t n_rhs;               /* evaluations of Hamilton's equations spent on this ray  */
} gp_ray_record;

/* One per ray when the disk is on, 48 bytes: crossing radius and redshift factor
 * g = (p.u_obs)/(p.u_emit) for a prograde circular Keplerian emitter (PAPER.md L356-374,
 * eq 56-57); unused slots hold NaN.                                                     */
typedef struct gp_disk_record {
  double r_cross[3];
  double g[3];
} gp_disk_record;

/* Device buffers, caller-owned.  rays: >= ray_count*sizeof(gp_ray_record), 32-byte
 * aligned.  disk: >= ray_count*sizeof(gp_disk_record) when max_crossings > 0 or the ring is on, else may be
 * NULL.  counters: >= 64 bytes, 8-byte aligned; the library zeroes it on the stream, uses
 * word 0 as the atomic work counter and leaves totals behind:
 *   [0] work counter (>= ray_count at exit)  [1] rays finished  [2] attempted steps
 *   [3] RHS evaluations
 *   [4] %globaltimer (ns) at kernel start   [5] when 99 % of the rays had finished (0 if never)
 *   [6] rays finished, counted live         [7] %globaltimer when the last block left
 * ([5]-[4] against [7]-[4] is the end-of-image tail of the persistent kernel.)                */
typedef struct gp_out_buffers {
  void *rays;
  size_t rays_bytes;
  void *disk;
  size_t disk_bytes;
  void *counters;
  size_t counters_bytes;
} gp_out_buffers;

/* ---- error codes (return values; per-ray failures are data, not errors) ------------- */
enum {
  GP_OK = 0,
  GP_E_BAD_METRIC = -1,
  GP_E_BAD_PARAM = -2,
  GP_E_NULL = -3,
  GP_E_SIZE = -4,
  GP_E_UNSUPPORTED = -5,
  GP_E_CUDA = -6,
  GP_E_STATIC_LIMIT = -7 /* gp_trace_static: ray_count > GP_STATIC_MAX_RAYS */
};

/* ---- entry points -------------------------------------------------------------------
 * All parameter structs are HOST memory, read before return.  `cuda_stream` is a
 * cudaStream_t passed as void* (NULL = the legacy default stream).  Unless stated, calls
 * validate synchronously, enqueue asynchronously on the stream and never synchronise.   */

/* The hot path (BASELINE.json north_star): trace camera->ray_count rays and write one
 * gp_ray_record (and gp_disk_record) per ray.  out->* are DEVICE pointers.
 * Returns GP_OK or a GP_E_* code.  On a validation error (every code but GP_E_CUDA) nothing has
 * been enqueued; GP_E_CUDA (the launch itself was refused) may leave the 64-byte memset of
 * `counters` enqueued.  Occupancy and SM count are cached per device id under a mutex: any
 * number of devices and host threads may call concurrently.                              */
int gp_trace(int metric_id, const gp_metric_params *metric, const gp_camera *camera,
             const gp_integrator_cfg *cfg, const gp_out_buffers *out, void *cuda_stream);

/* Same computation with HOST output buffers (out->* are host pointers, pinned or
 * pageable; counters may be NULL).  Pinned (page-locked, mapped) rays / disk buffers are written
 * by the kernel itself, record by record as the rays end, so the transfer overlaps the tracing;
 * pageable buffers are staged through device scratch from a library-owned stream-ordered pool and
 * copied back.  Either way the stream is SYNCHRONISED before returning.  This is the end-to-end
 * call bench.py times.  Re-entrant: the 64-byte device counters (and the staging scratch) are
 * allocated per call, stream-ordered, from a library-owned pool that exists once per device
 * (created under a mutex on first use, kept for the life of the process), so concurrent calls
 * on different streams, host threads and devices are independent.                               */
int gp_trace_host(int metric_id, const gp_metric_params *metric, const gp_camera *camera,
                  const gp_integrator_cfg *cfg, const gp_out_buffers *out, void *cuda_stream);

/* gp_trace for callers that may not allocate (code under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc).  Same kernels, same records, same validation and error behaviour as gp_trace;
 * the difference is where the scratch lives.  gp_trace takes its work counter from the caller's
 * `counters` block and, with cfg.segment_steps != 0, two slot lists from a stream-ordered pool; here
 * both sit in ONE file-scope `static __device__` array of the library (128 bytes of counters and list
 * counts + 2 x GP_STATIC_MAX_RAYS x 8 bytes of lists = 16 MiB + 128 bytes, which every GPU that loads
 * the library holds until the process exits).  The call makes no cudaMalloc / cudaFree / pool
 * allocation: it enqueues memsets of the 128 bytes that must start at zero (the lists need no clearing,
 * only the first `count` entries of a list are ever read), the launches, and one 64-byte
 * device-to-device copy if out->counters is given.
 *   out->rays, out->disk  DEVICE, as for gp_trace (sizes and alignment checked the same way).
 *   out->counters         DEVICE, >= 64 bytes, 8-byte aligned, or NULL: receives a copy of the totals
 *                         ([0]..[7] as documented at gp_out_buffers) after the last launch.
 *   camera->ray_count     <= GP_STATIC_MAX_RAYS, else GP_E_STATIC_LIMIT and nothing is enqueued (tile a
 *                         larger image with ray_begin / ray_count, one call per tile, or use gp_trace).
 * NOT re-entrant per device: every call on a device shares the array, which keeps the previous call's
 * contents until this call's memsets run.  Calls on the SAME stream are ordered and correct; calls that
 * overlap on the GPU (different streams without an event between them, or several host threads on one
 * device) race on the work counter and produce garbage.  Different devices hold different copies and
 * are independent; the array's device address is looked up once per device, under a mutex, with that
 * device current.                                                                                  */
int gp_trace_static(int metric_id, const gp_metric_params *metric, const gp_camera *camera,
                    const gp_integrator_cfg *cfg, const gp_out_buffers *out, void *cuda_stream);

/* Steps a2+a3 alone (pixel -> (alpha,beta) -> initial state), for inspection and parity.
 * states8: DEVICE, ray_count*8 doubles (t, r, theta, phi, p_t, p_r, p_theta, p_phi).
 * alpha_beta2: DEVICE, ray_count*2 doubles, or NULL.                                    */
int gp_init_conditions(int metric_id, const gp_metric_params *metric, const gp_camera *camera,
                       void *states8, size_t states_bytes, void *alpha_beta2, size_t ab_bytes,
                       void *cuda_stream);

/* Step a4 alone: inverse metric and its r, theta derivatives at n points.
 * r_theta2: DEVICE, n*2 doubles (r, theta).  out15: DEVICE, n*15 doubles in the order
 * g^tt, g^tphi, g^phiphi, g^rr, g^thth, then the same five d/dr, then the same five
 * d/dtheta.  Closed form for Schwarzschild and Kerr, forward-mode duals for MN.         */
int gp_eval_metric(int metric_id, const gp_metric_params *metric, const void *r_theta2,
                   int64_t n, void *out15, size_t out_bytes, void *cuda_stream);

/* One evaluation of Hamilton's equations (steps a4+a5) at n states.
 * states8: DEVICE n*8 doubles as above.  rhs6: DEVICE n*6 doubles
 * (dt, dr, dtheta, dphi, dp_r, dp_theta)/dlambda.                                       */
int gp_eval_rhs(int metric_id, const gp_metric_params *metric, const void *states8, int64_t n,
                void *rhs6, size_t rhs_bytes, void *cuda_stream);

/* FP64 FMA peak probe used for the roofline denominator: every thread of a full-chip grid
 * runs `iters` rounds of 8 independent dependent-chain DFMAs; scratch (DEVICE, >= 8 bytes)
 * receives a value that keeps the chain alive.  *flops_out (HOST) = 2 * DFMAs issued.
 * Time it with events on the stream.                                                    */
int gp_probe_fp64_fma(int64_t iters, void *scratch, size_t scratch_bytes, double *flops_out,
                      void *cuda_stream);

/* ---- image formation (the drawing script's kernel that
 * maps "output positions" to colours) -------
 * One RGBA8 pixel per image pixel from the ray records of a finished trace of the same camera
 * (ray = (j*S + sj)*W*S + (i*S + si), S = supersample; the S*S sub-ray colours are averaged).
 * Per sub-ray, in FP64 with individually rounded operations (bit-exact against any IEEE-754
 * implementation of the same formulas):
 *   status != ESCAPED : shadow colour (0,0,0); in mode 2 (0,1,1) (cyan).
 *   otherwise canonicalise the raw exit angles without transcendentals:
 *     th = theta - 2pi*floor(theta/2pi); ph = phi; if (th > pi) { th = 2pi - th; ph = ph + pi; }
 *     ph = ph - 2pi*floor(ph/2pi);
 *   mode 0 (celestial grid, L404): base colour PALETTE8[4*(th >= pi/2) + min(3, floor(ph/(pi/2)))];
 *     a point within grid_half_width_deg of a multiple of grid_step_deg in th or in ph takes the
 *     line colour (0.05, 0.05, 0.05).
 *   mode 1 (background texture with bilinear filtering, L422; procedural stand-in for the ESO
 *     panorama): equirectangular tex_width x tex_height texels, texel (i, j) = the three low bytes
 *     of SplitMix64(tex_seed * 0x9E3779B97F4A7C15 + j * tex_width + i) / 255; sample at
 *     u = ph/(2pi)*tex_width - 0.5 (wrapping), v = th/pi*tex_height - 0.5 (clamped).
 *   mode 2 (exit-time bands, L430): PALETTE6[floor(|t| / time_period) mod 6].
 *   disk overlay (L735; needs `disk`; takes precedence over everything above, the disk is opaque; a ray that
 *     ended on the solid ring, status HIT_RING, carries its hit in the same slot and is coloured the same way):
 *     if the first recorded crossing exists (r_cross[0] is not NaN), the colour is
 *     g < 1: blue (0.1,0.2,1) -> white by (g - g_lo)/(1 - g_lo);  g >= 1: white -> red (1,0.1,0.1)
 *     by (g - 1)/(g_hi - 1), both parameters clamped to [0, 1].
 *   pixel byte = floor(255 * mean + 0.5), alpha = 255.
 * PALETTE8 = (.85,.25,.25) (.25,.75,.25) (.25,.35,.9) (.9,.8,.2) (.55,.15,.15) (.15,.45,.15)
 * (.15,.2,.6) (.6,.5,.1); PALETTE6 = (.9,.1,.1) (.9,.6,.1) (.8,.9,.1) (.1,.8,.2) (.1,.5,.9) (.6,.1,.9).
 * rays: DEVICE, n = W*H*S*S gp_ray_record; disk: DEVICE n gp_disk_record or NULL (required when
 * disk_overlay != 0); rgba8: DEVICE, W*H*4 bytes, row j = 0 first.  HBM-bound: reads 128 (+48) bytes
 * per sub-ray, writes 4 bytes per pixel.  GP_E_BAD_PARAM on non-positive sizes, unknown mode,
 * non-positive grid / period / texture sizes for the mode in use, g_lo >= 1 or g_hi <= 1.        */
typedef struct gp_shade_cfg {
  int32_t width, height, supersample;
  int32_t mode;                 /* 0 celestial grid, 1 procedural texture, 2 exit-time bands */
  double grid_step_deg, grid_half_width_deg;
  int32_t tex_width, tex_height;
  uint64_t tex_seed;
  double time_period;
  int32_t disk_overlay;         /* 0 off, 1 colour the first recorded disk crossing by g     */
  int32_t reserved_;
  double g_lo, g_hi;
} gp_shade_cfg;

/* Alignment (GP_E_BAD_PARAM otherwise): rays 16 bytes (128-bit loads; the buffers gp_trace accepts are
 * 32-byte aligned), disk 8 bytes, rgba8 4 bytes (one 32-bit store per pixel).                      */
int gp_shade(const gp_shade_cfg *cfg, const void *rays, size_t rays_bytes, const void *disk,
             size_t disk_bytes, void *rgba8, size_t rgba_bytes, void *cuda_stream);

/* ---- orbits from explicit initial states (section 3.2.1 and Fig 1: time-like
 * test orbits, the same equations with H = -1/2; L719, Fig 11: neighbouring null orbits; SURVEY.md
 * section 8(f) NEXT-3) --------------------------------------------------------------------------
 * Integrates n states (t, r, theta, phi, p_t, p_r, p_theta, p_phi; any value of H) with the
 * Dormand-Prince pair and the controller of scheme 2 from lambda = 0 to lambda_end, every attempted
 * step being min(h, h_max, lambda_next - lambda) so that the state is sampled exactly at
 * lambda_k = (k+1) lambda_end / n_samples, k < n_samples; a step cut short by a sample time keeps
 * the controller's previous proposal when that is larger; the first proposal is h0.
 * states8: DEVICE n*8 doubles.  samples: DEVICE n*n_samples*8 doubles, per sample
 * (t, r, theta, phi, p_r, p_theta, 2H, lambda), NaN after an orbit ended early.  status: DEVICE n
 * uint32 (GP_RAY_ESCAPED = reached lambda_end, GP_RAY_CAPTURED = r < r_H (1 + eps_capture),
 * GP_RAY_MAXSTEPS, GP_RAY_STEP_UNDERFLOW).  n_steps: DEVICE n uint64 attempted steps.
 * GP_E_BAD_PARAM on non-positive rtol, h0, h_max, lambda_end, n_samples, negative atol / max_steps,
 * and on misaligned buffers: samples must be 32-byte aligned (written with 256-bit stores), states8 and
 * n_steps 8-byte, status 4-byte.                                                                      */
typedef struct gp_orbit_cfg {
  double rtol, atol, h0, h_max, lambda_end, eps_capture;
  int64_t n_samples, max_steps;
} gp_orbit_cfg;

int gp_integrate_orbits(int metric_id, const gp_metric_params *metric, const gp_orbit_cfg *cfg,
                        const void *states8, int64_t n, void *samples, size_t samples_bytes, void *status,
                        size_t status_bytes, void *n_steps, size_t n_steps_bytes, void *cuda_stream);

/* Horizon radius r_H and prograde ISCO radius used by the library for these parameters
 * (r_isco = NaN for GP_MANKO_NOVIKOV).  Host-only helper.                               */
int gp_metric_radii(int metric_id, const gp_metric_params *metric, double *r_horizon,
                    double *r_isco);

size_t gp_ray_record_size(void);  /* 128 */
size_t gp_disk_record_size(void); /* 48  */
size_t gp_counters_size(void);    /* 64  */
int64_t gp_static_max_rays(void); /* GP_STATIC_MAX_RAYS */
int gp_version(void);
/* Static string for a GP_E_* code; for GP_E_CUDA the last CUDA error text seen by this
 * thread is appended.                                                                   */
const char *gp_strerror(int code);

#ifdef __cplusplus
} /* extern "C" */
#endif

#endif /* GP_H_ */
