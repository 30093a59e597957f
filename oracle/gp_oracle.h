/* gp_oracle.h — TEST INFRASTRUCTURE, not the product.
 *
 * Plain, slow, scalar double-precision CPU implementation of the null-geodesic hot path,
 * written from PAPER.md (arXiv 2310.15183) and the readings listed in DESIGN.md section 3.
 * It shares no code, header, table or helper with the CUDA library (include/gp.h,
 * paper_2310_15183_b200/csrc); its structs are declared here independently.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * Pins (tests/test_oracle_*.py, tests/test_golden_closed_forms.py, all `-m "not gpu"`): flat-space closed
 * form, Schwarzschild critical impact parameter and deflection quadrature, Kerr radial-potential classifier
 * and Bardeen's critical curve, Carter constant, photon-orbit and ISCO radii, Manko-Novikov -> Kerr at
 * q = 0, Manko-Novikov vacuum (Ernst) equations, the Manko-Novikov inverse metric against a 50-digit mpmath
 * evaluation of eq 20-39, equatorial mirror symmetry, Dormand-Prince order conditions, the step-size
 * controller and error norm re-enacted from the published tableau (test_oracle_controller_pin.py), scipy
 * DOP853 trajectories, eq 56 against the closed-form Keplerian emitter and a dynamic circular-orbit check,
 * the solid ring against a brute-force straight-line entry search in flat space, its thin limit and mirror
 * symmetry (test_oracle_ring_pins.py), the image-formation oracle against a vectorised restatement of
 * the contract text (test_oracle_shade_contract.py).
 * Parity unpinned: exit angles inside Manko-Novikov chaotic sets, any state of a MAXSTEPS ray, and the exit
 * state of Manko-Novikov CAPTURED rays that the rounding probe flags (statistical / status-only comparison;
 * DESIGN.md section 5, R21, R24).
 */
#ifndef GP_ORACLE_H_
#define GP_ORACLE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* metric ids: 0 Schwarzschild (eq 8), 1 Kerr Boyer-Lindquist (eq 9-14), 2 Manko-Novikov (eq 20-39) */
typedef struct orc_metric {
  int32_t id;
  int32_t pad_;
  double M, a, q;
} orc_metric;

typedef struct orc_camera {
  double r_obs, theta_obs, phi_obs;
  double alpha_min, alpha_max, beta_min, beta_max;
  int64_t width, height, supersample;
  uint64_t jitter_seed;
  double jitter_amp_px, shift_x_px, shift_y_px;
  /* 0: pinhole in the ZAMO tetrad (BASELINE.json); 1: the paper's Euclidean screen:
   * start points alpha e_phi + beta e_up on a flat screen centred at r_obs c_hat, directions
   * -c_hat + focal_2f_over_d (alpha e_phi + beta e_up) (0 = parallel rays, "focal distance infinity") */
  int64_t projection;
  double focal_2f_over_d;
} orc_camera;

typedef struct orc_cfg {
  int64_t scheme; /* 0 RK4 fixed h; 1 RK4 h = h_rel*r; 2 Dormand-Prince 5(4) adaptive */
  double h, h_rel, rtol, atol, h_cap_rel;
  int64_t max_steps;
  double lambda_max;
  double eps_capture, r_escape;
  double disk_r_in, disk_r_out;
  int64_t max_crossings;
  /* > 0: a solid ring (Fig 15-17: "a region in space around the equator of non-zero
   * thickness", hit when "the ray propagat[es] to a point inside the volume"): the set
   * disk_r_in <= r <= disk_r_out, |theta - pi/2| <= ring_half_angle.  Opaque: the ray ends there with
   * status 5, located on the face it entered through (see trace_ray); disk_r[0], disk_g[0] = hit radius
   * and redshift factor of the circular equatorial emitter at that radius.  Needs max_crossings = 0;
   * every scheme (the landing steps use the scheme's own formula, R14). */
  double ring_half_angle;
} orc_cfg;

/* status: 0 escaped, 1 captured, 2 max steps, 3 non-finite, 4 step underflow, 5 hit the ring */
typedef struct orc_record {
  int64_t status, n_accepted, n_rejected, n_equator_crossings, n_disk_recorded, n_rhs;
  double alpha, beta;
  double t, r, theta, phi, p_t, p_r, p_theta, p_phi, lambda;
  double h_max, q_drift, sin_theta_min, err_margin;
  double disk_r[3], disk_g[3];
} orc_record;

/* O1: ray index -> image-plane point (R11) */
void orc_alpha_beta(const orc_camera *cam, int64_t ray, double *alpha, double *beta);
/* covariant metric: out5 = g_tt, g_tphi, g_phiphi, g_rr, g_thth */
int orc_metric_cov(const orc_metric *m, double r, double theta, double *out5);
/* inverse metric and r, theta derivatives: out15 = (g^tt, g^tphi, g^phiphi, g^rr, g^thth), d/dr, d/dtheta */
int orc_metric_inv(const orc_metric *m, double r, double theta, double *out15);
/* same, every derivative by the complex-step method on the inverse of the covariant metric */
int orc_metric_inv_complex_step(const orc_metric *m, double r, double theta, double *out15);
/* Manko-Novikov potentials: out = f, omega, e^{2 gamma}, A, B, C, a_frak, b_frak, psi, gamma' */
int orc_mn_potentials(const orc_metric *m, double r, double theta, double *out10);
/* O2+O3: initial state8 = t, r, theta, phi, p_t, p_r, p_theta, p_phi */
int orc_initial_state(const orc_metric *m, const orc_camera *cam, double alpha, double beta,
                      double *state8);
/* O4: Hamilton's equations, rhs6 = d(t, r, theta, phi, p_r, p_theta)/dlambda */
int orc_rhs(const orc_metric *m, const double *state8, double *rhs6);
/* horizon radius and prograde ISCO (NaN for Manko-Novikov) */
int orc_radii(const orc_metric *m, double *r_horizon, double *r_isco);
/* prograde Keplerian emitter: Omega_K, u^t, and g for a ray with constants (p_t, p_phi) */
int orc_kepler(const orc_metric *m, double r, double p_t, double p_phi, double *out3);
/* the same from eq 56 solved with the metric's own d_r g^{mu nu} (any metric) */
int orc_kepler_general(const orc_metric *m, double r, double p_t, double p_phi, double *out3);
/* Dormand-Prince tableau: c[7], a[7*7] (row-major, lower triangle), b5[7], e[7] */
void orc_dp54_tableau(double *c7, double *a49, double *b7, double *e7);
/* one explicit step of scheme (0/1: RK4, 2: DP5(4)) from state8 with step h, for tests:
 * out_state8, err (scheme 2, else 0) */
int orc_single_step(const orc_metric *m, int64_t scheme, const double *state8, double h,
                    double rtol, double atol, double *out_state8, double *err);
/* O5-O8: trace rays ray_begin + k*ray_stride, k < ray_count; out[k]; OpenMP over rays with
 * n_threads threads (<= 0: all).  Returns the number of threads used, < 0 on bad arguments. */
int orc_trace(const orc_metric *m, const orc_camera *cam, const orc_cfg *cfg, int64_t ray_begin,
              int64_t ray_count, int64_t ray_stride, orc_record *out, int n_threads);
/* trace one ray given (alpha, beta) directly; optional trajectory dump of accepted states:
 * path (n_path_max * 8 doubles: lambda, t, r, theta, phi, p_r, p_theta, h), *n_path written */
int orc_trace_one(const orc_metric *m, const orc_camera *cam, const orc_cfg *cfg, double alpha,
                  double beta, orc_record *out, double *path, int64_t n_path_max, int64_t *n_path);

/* ---- orbits from explicit initial states (section 3.2.1: time-like test orbits with
 * H = -1/2; Fig 11: neighbouring null orbits).  The same Hamilton's equations and the same
 * Dormand-Prince pair, integrated to lambda_end with the state sampled at lambda_k = (k+1) lambda_end /
 * n_samples: every attempted step is min(h, h_max, lambda_next - lambda); a step cut short by a sample
 * time keeps the controller's previous proposal when that is larger.  samples: n * n_samples * 8
 * doubles (t, r, theta, phi, p_r, p_theta, 2H, lambda), NaN after an orbit ended early; status per
 * orbit: 0 reached lambda_end, 1 captured (r < r_H (1 + eps_capture)), 2 step budget, 4 step underflow. */
typedef struct orc_orbit_cfg {
  double rtol, atol, h0, h_max, lambda_end, eps_capture;
  int64_t n_samples, max_steps;
} orc_orbit_cfg;
int orc_integrate_orbits(const orc_metric *m, const orc_orbit_cfg *cfg, const double *states8, int64_t n,
                         double *samples, int64_t *status, int64_t *n_steps);

#ifdef __cplusplus
}
#endif
#endif
