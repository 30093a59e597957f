// gp_camera.cuh — SURVEY.md section 8 rows a2 (ray index -> image-plane point) and a3 (pinhole
// direction in the observer's ZAMO tetrad -> covariant momentum with H = 0).
//
// Replaces the Euclidean screen of PAPER.md L314-348 (section 3.3.1, eq 51-55) as BASELINE.json
// prescribes; DESIGN.md section 3 readings R11 (pixel map, jitter generator) and R12 (time-
// reversed ray, unit locally measured energy).  Row a2 is evaluated with individually rounded
// operations (__dadd_rn/__dmul_rn/__ddiv_rn never contract into FMAs), so alpha and beta are
// bit-identical to any IEEE-754 double implementation of the same formula.
#ifndef GP_CAMERA_CUH_
#define GP_CAMERA_CUH_

#include <stdint.h>

namespace gp {

struct CameraConst {
  // pixel map (R11)
  double alpha_min, beta_min;
  double dalpha, dbeta;          // (alpha_max-alpha_min)/width, (beta_max-beta_min)/height
  double supersample_d;          // (double)S
  double jitter_amp_px, shift_x_px, shift_y_px;
  unsigned long long jitter_seed;
  long long Wt;                  // width * S
  double inv_Wt;                 // 1 / Wt (seed of the row / column split of the ray index)
  double inv_S;                  // 1 / S when S is a power of two (the division by S is then an exact
                                 // multiplication), else 0: IEEE division
  long long ray_begin, ray_count, ray_stride;
  // observer (R12): position and ZAMO tetrad constants from the covariant metric there
  double r_obs, theta_obs, phi_obs;
  double sq_grr, sq_gthth, sq_gpp; // sqrt(g_rr), sqrt(g_thth), sqrt(g_phiphi)
  double inv_zeta;                 // sqrt(-(g_tt + Omega g_tphi))
  double Omega;                    // -g_tphi/g_phiphi
  // projection = 1 (the paper's Euclidean screen): frame and focal factor
  int projection;
  int metric_id;
  double k2;                       // 2f/d
  double a_cam;                    // spin used by eq 51-53 (0 for Schwarzschild)
  double chat[3], eph[3], eup[3];  // screen normal (towards the observer) and its two axes
};

#if defined(__CUDACC__)

// SplitMix64 finaliser (Steele, Lea & Flood 2014), keyed statelessly by (seed, ray, axis).
__device__ __forceinline__ double jitter_unit(unsigned long long seed, unsigned long long ray,
                                              unsigned long long axis) {
  unsigned long long z = seed * 0x9E3779B97F4A7C15ULL + 2ULL * ray + axis;
  z += 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  z = z ^ (z >> 31);
  return __dmul_rn((double)(z >> 11), 1.0 / 9007199254740992.0);  // exact: 53-bit integer x 2^-53
}

// Row a2.  ray = index in the supersampled image, row-major, J = 0 <-> beta_min.
__device__ __forceinline__ void alpha_beta(const CameraConst &cc, long long ray, double &alpha,
                                           double &beta) {
  // row J = ray div Wt, column I = ray mod Wt: quotient estimated in FP64 (exact to +-1 for ray < 2^52),
  // corrected with integers — a 64-bit integer division is ~80 instructions, once per ray
  long long J = (long long)__dmul_rn((double)ray, cc.inv_Wt);
  long long I = ray - J * cc.Wt;
  if (I < 0) { J -= 1; I += cc.Wt; }
  else if (I >= cc.Wt) { J += 1; I -= cc.Wt; }
  double jx = 0.0, jy = 0.0;
  if (cc.jitter_amp_px > 0.0) {
    double ux = jitter_unit(cc.jitter_seed, (unsigned long long)ray, 0ULL);
    double uy = jitter_unit(cc.jitter_seed, (unsigned long long)ray, 1ULL);
    jx = __dmul_rn(__dadd_rn(__dmul_rn(2.0, ux), -1.0), cc.jitter_amp_px);
    jy = __dmul_rn(__dadd_rn(__dmul_rn(2.0, uy), -1.0), cc.jitter_amp_px);
  }
  // (I + 0.5)/S: S = 2^k makes x * (1/S) the same double as x / S
  double xs = __dadd_rn((double)I, 0.5), ys = __dadd_rn((double)J, 0.5);
  if (cc.inv_S != 0.0) {
    xs = __dmul_rn(xs, cc.inv_S);
    ys = __dmul_rn(ys, cc.inv_S);
  } else {
    xs = __ddiv_rn(xs, cc.supersample_d);
    ys = __ddiv_rn(ys, cc.supersample_d);
  }
  double X = __dadd_rn(__dadd_rn(xs, jx), cc.shift_x_px);
  double Y = __dadd_rn(__dadd_rn(ys, jy), cc.shift_y_px);
  alpha = __dadd_rn(cc.alpha_min, __dmul_rn(X, cc.dalpha));
  beta = __dadd_rn(cc.beta_min, __dmul_rn(Y, cc.dbeta));
}

// Row a3.  Tetrad tangent of the traced (time-reversed) ray is (-1, n) with the pinhole direction
// n = (-r_o, -beta, +alpha)/D in the (r, theta, phi) legs; lowering with the tetrad gives
// p_r = sqrt(g_rr) n_r, p_th = sqrt(g_thth) n_th, p_ph = sqrt(g_phiphi) n_ph,
// p_t = 1/zeta - Omega p_ph, and H = 0 by construction.
__device__ __forceinline__ void initial_momentum(const CameraConst &cc, double alpha, double beta,
                                                 double &pt, double &pr, double &pth, double &pph) {
  double ro = cc.r_obs;
  double iD = rsqrt(ro * ro + alpha * alpha + beta * beta);
  pr = cc.sq_grr * (-ro * iD);
  pth = cc.sq_gthth * (-beta * iD);
  pph = cc.sq_gpp * (alpha * iD);
  pt = cc.inv_zeta - cc.Omega * pph;
}

#endif  // __CUDACC__

}  // namespace gp
#endif
