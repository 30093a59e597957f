// gp_math.cuh — FP64 elementary functions for the tracer's inner loop, written for the sm_100a
// issue model.
//
// Why not the CUDA math library here: profiles/trace_dp54_r01a.md showed that 28 % of the warp
// instructions of the first trace_dp54 were UMOV/IMAD.MOV pairs materialising 64-bit literals (the
// library's sincos, division and pow carry their coefficients as immediates), and that each `a / b`
// and each fmax drags a denormal / NaN slow-path test through the instruction stream.  On sm_100a
// an FP64 instruction holds the issue slot for two cycles and every other instruction costs a full
// cycle on top, so those instructions cost as much as the arithmetic.
// Every literal below lives in __constant__ memory (one LDCU per use at worst, 128-bit pairs where
// adjacent); every function is branch-free on the range the integrator produces and falls back to
// the library outside it.
//
// Accuracy: sincos polynomial error 1e-17 / 5e-19 before rounding, rcp_nr and div_nr <= 1 ulp,
// pow_m1_5 <= 2 ulp; exercised against the oracle by tests/test_gpu_parity.py
// (test_eval_rhs_matches_oracle, test_eval_metric_matches_oracle and every trace test).
#ifndef GP_MATH_CUH_
#define GP_MATH_CUH_

#include <math.h>

#if defined(__CUDACC__)
#define GP_HD __host__ __device__ __forceinline__
#else
#define GP_HD inline
#endif

namespace gp {

#if defined(__CUDACC__)

// Coefficients are near-minimax fits made for this file (Chebyshev-node interpolation of
// (sin r / r - 1)/r^2 and (cos r - 1 + r^2/2)/r^4 on r^2 <= 1.02 (pi/4)^2, 60-digit mpmath).
struct MathConst {
  double two_over_pi;
  double pio2_hi, pio2_mid, pio2_lo;  // pi/2 split 33 + 33 + 53 bits: q*hi and q*mid are exact for |q| < 2^20
  double s[6];                        // sin: r + r z (s0 + s1 z + ... + s5 z^5), z = r^2
  double c[6];                        // cos: 1 - z/2 + z^2 (c0 + ... + c5 z^5)
  double one, half, fifth, six_fifths;
  double magic;
  double as[6];                       // sin d = d + d z (as0 + ... + as4 z^4), z = d^2: Taylor (as5 unused)
  double ac[7];                       // cos d - 1 = z (ac0 + ... + ac5 z^5) (ac6 unused)
};

__constant__ MathConst kMath = {
    0x1.45f306dc9c883p-1,
    0x1.921fb54400000p+0, 0x1.0b4611a600000p-34, 0x1.3198a2e037073p-69,
    {-0x1.5555555555555p-3, 0x1.1111111110b23p-7, -0x1.a01a019e623afp-13, 0x1.71de376b9c575p-19,
     -0x1.ae5fdeb852566p-26, 0x1.5dfb4dfaf15abp-33},
    {0x1.5555555555555p-5, -0x1.6c16c16c1691fp-10, 0x1.a01a019f3df42p-16, -0x1.27e4fa025e03dp-22,
     0x1.1eeb52bea9072p-29, -0x1.906dd38cb66a1p-37},
    1.0, 0.5, 0.2, 1.2, 6755399441055744.0,
    {-0x1.5555555555555p-3, 0x1.1111111111111p-7, -0x1.a01a01a01a01ap-13, 0x1.71de3a556c734p-19, -0x1.ae64567f544e4p-26, 0x1.6124613a86d09p-33},
    {-0x1.0000000000000p-1, 0x1.5555555555555p-5, -0x1.6c16c16c16c17p-10, 0x1.a01a01a01a01ap-16, -0x1.27e4fb7789f5cp-22, 0x1.1eed8eff8d898p-29, -0x1.93974a8c07c9dp-37}};

// max / min of two doubles without fmax's NaN canonicalisation: a NaN candidate never replaces
// the running value (the same outcome fmax(running, NaN) gives).
__device__ __forceinline__ double dmax(double run, double cand) { return cand > run ? cand : run; }
__device__ __forceinline__ double dmin(double run, double cand) { return cand < run ? cand : run; }

// 1/x to about 1 ulp for normal finite x: MUFU.RCP64H seed (relative error e0 <= 2^-20) + one cubic
// Newton step, y (1 + e + e^2) = (1/x)(1 - e^3): e0^3 <= 2^-60 is 1/128 ulp, so what is left is the
// rounding of the last FMA.  (A second, quadratic step — two more DFMAs, kept through round 1 — only
// turned <= 1.5 ulp into <= 1 ulp; dropping it bought 1.4 % on the headline.)  x = 0 or non-finite
// gives a non-finite result (the integrator's finite tests catch it); subnormal x is outside the
// integrator's range.
__device__ __forceinline__ double rcp_nr(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);   // 1.0 travels as an immediate operand (upper word only)
  e = fma(e, e, e);
  return fma(y, e, y);
}

// 1/sqrt(x) to about 1 ulp for normal finite x > 0: MUFU.RSQ64H seed (relative error e0 ~ 2^-22) + one cubic
// Newton step, y (1 + e/2 + 3 e^2/8) with e = 1 - x y^2: what is left is e0^3 and the rounding of the last FMA.
__device__ __forceinline__ double rsqrt_nr(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-(x * y), y, 1.0);
  double p = fma(0.375, e, 0.5);
  return fma(y * e, p, y);
}

// a/b to <= 1 ulp given y = rcp_nr(b): one residual correction.
__device__ __forceinline__ double div_nr(double a, double b, double y) {
  double q = a * y;
  double rem = fma(-b, q, a);
  return fma(rem, y, q);
}

// sin and cos of x for |x| < 1e5 (the polar angle never leaves a few multiples of pi); the
// library routine takes over beyond that.  Cody-Waite reduction to |r| <= pi/4 with a three-part
// pi/2, then the two kernels, then the quadrant swap.
__device__ __noinline__ double2 sincos_library(double x) {
  double2 r;
  sincos(x, &r.x, &r.y);
  return r;   // by value: the results come back in registers, not through the caller's stack frame
}

__device__ __forceinline__ void sincos_fast(double x, double *sn, double *cs) {
  if (!(fabs(x) < 1.0e5)) {
    double2 sc = sincos_library(x);
    *sn = sc.x;
    *cs = sc.y;
    return;
  }
  double qd = rint(x * kMath.two_over_pi);
  int q = __double2int_rn(qd);
  double r = fma(-qd, kMath.pio2_hi, x);
  r = fma(-qd, kMath.pio2_mid, r);
  r = fma(-qd, kMath.pio2_lo, r);
  double z = r * r;
  double ps = fma(z, kMath.s[5], kMath.s[4]);
  double pc = fma(z, kMath.c[5], kMath.c[4]);
  ps = fma(z, ps, kMath.s[3]);
  pc = fma(z, pc, kMath.c[3]);
  ps = fma(z, ps, kMath.s[2]);
  pc = fma(z, pc, kMath.c[2]);
  ps = fma(z, ps, kMath.s[1]);
  pc = fma(z, pc, kMath.c[1]);
  ps = fma(z, ps, kMath.s[0]);
  pc = fma(z, pc, kMath.c[0]);
  double sr = fma(r * z, ps, r);                              // sin r
  double cr = fma(z * z, pc, fma(-0.5, z, 1.0)); // cos r
  // quadrant: q mod 4 = 0: (s, c); 1: (c, -s); 2: (-s, -c); 3: (-c, s)
  double a = (q & 1) ? cr : sr;
  double b = (q & 1) ? sr : cr;
  // sign flips on the high word (one LOP3 each) instead of FP64 negate + select
  *sn = __hiloint2double(__double2hiint(a) ^ ((q & 2) << 30), __double2loint(a));
  *cs = __hiloint2double(__double2hiint(b) ^ (((q + 1) & 2) << 30), __double2loint(b));
}

// sin and cos of (theta_n + d) from sn = sin theta_n, cn = cos theta_n by the addition theorems, for the
// stage angles of one Runge-Kutta attempt (|d| = |step x sum a_ij dtheta/dlambda|, a few hundredths of a
// radian in practice).  Taylor kernels through d^11 / d^12: truncation below 3e-18 for |d| <= 1/4 and
// 2e-14 at |d| = 1/2 (one more term each bought nothing at any tolerance the integrator is asked for and
// cost 1.6 % of the headline).  No range reduction, no quadrant logic, no branch: 18 FP64 instructions and
// nothing else, against 21 + 16 for sincos_fast.  A wild trial step (|d| > 1/2) gets a finite wrong value; its error estimate is then
// huge and the step is rejected (R10 item 2), which is what happens to such a step anyway.
__device__ __forceinline__ void sincos_add(double sn, double cn, double d, double *s, double *c) {
  double z = d * d;
  // The three highest coefficients are rounded to their upper 32 bits so that they travel as immediate
  // operands of the DFMA (no constant load): a relative change of 2.3e-7 in terms that are themselves below
  // 3e-13 of the result for |d| <= 1/4.
  double ps = fma(z, -0x1.ae64500000000p-26, kMath.as[3]);
  double pc = fma(fma(z, 0x1.1eed900000000p-29, -0x1.27e5000000000p-22), z, kMath.ac[3]);
  ps = fma(z, ps, kMath.as[2]);
  pc = fma(z, pc, kMath.ac[2]);
  ps = fma(z, ps, kMath.as[1]);
  pc = fma(z, pc, kMath.ac[1]);
  ps = fma(z, ps, kMath.as[0]);
  pc = fma(z, pc, kMath.ac[0]);
  double sd = fma(d * z, ps, d);   // sin d
  double cm = z * pc;              // cos d - 1
  *s = fma(sn, cm, fma(cn, sd, sn));
  *c = fma(cn, cm, fma(-sn, sd, cn));
}

// FP32 form for the single-precision and mixed variants: Taylor through d^7 / d^8 (truncation 4e-11 at
// |d| = 1/4, below half an FP32 ulp).
__device__ __forceinline__ void sincos_add(float sn, float cn, float d, float *s, float *c) {
  float z = d * d;
  float ps = fmaf(z, fmaf(z, -1.98412698e-4f, 8.33333333e-3f), -1.66666667e-1f);
  float pc = fmaf(z, fmaf(z, fmaf(z, 2.48015873e-5f, -1.38888889e-3f), 4.16666667e-2f), -0.5f);
  float sd = fmaf(d * z, ps, d);
  float cm = z * pc;
  *s = fmaf(sn, cm, fmaf(cn, sd, sn));
  *c = fmaf(cn, cm, fmaf(-sn, sd, cn));
}

// x^(-1/5) for x in [1e-5, 1e4] (the controller clamps outside, R10 item 3): FP32 seed from the
// SFU (lg2/ex2, about 1e-6 relative), two Newton steps on y^-5 = x (error 3 e^2 per step) -> <= 2 ulp.
// (One step, 1e-12 relative, saves 0.7 % of the headline's time and keeps every exit state within
// 1e-9, but moves the step sequence enough that the rounding-level max|H| of one Manko-Novikov ray
// in 8557 left the 25 % band of tests/parity_rules.py: measured at the end of round 1, not kept.)
__device__ __forceinline__ double pow_m1_5(double x) {
  float xf = __double2float_rn(x), lg, yf;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lg) : "f"(xf));
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(yf) : "f"(-0.2f * lg));
  {
    float y2 = yf * yf, y5 = y2 * y2 * yf;
    float e = fmaf(-xf, y5, 1.0f);
    yf = fmaf(yf * 0.2f, e, yf);
  }
  double y = (double)yf;
#pragma unroll
  for (int i = 0; i < 1; ++i) {
    double y2 = y * y;
    double y5 = y2 * y2 * y;
    double e = fma(-x, y5, 1.0);
    y = fma(y * kMath.fifth, e, y);
  }
  return y;
}

// The same with the range clamp applied to the FP32 seed only (two FMNMX): for x outside [1e-5, 1e4] the
// result is not x^(-1/5) but it stays on the same side of the controller's clamps (> 5.6 below, < 0.16 or
// negative above), which is all that is used of it there.
__device__ __forceinline__ double pow_m1_5_clamped(double x) {
  float xf = fminf(fmaxf(__double2float_rn(x), 1.0e-5f), 1.0e4f), lg, yf;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lg) : "f"(xf));
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(yf) : "f"(-0.2f * lg));
  {
    float y2 = yf * yf, y5 = y2 * y2 * yf;
    float e = fmaf(-xf, y5, 1.0f);
    yf = fmaf(yf * 0.2f, e, yf);
  }
  double y = (double)yf;
  double y2 = y * y;
  double y5 = y2 * y2 * y;
  double e = fma(-x, y5, 1.0);
  return fma(y * kMath.fifth, e, y);
}

#endif  // __CUDACC__

// The same source serves the device (fast forms above) and the host (observer constants, row a3).
GP_HD double frcp(double x) {
#if defined(__CUDA_ARCH__)
  return rcp_nr(x);
#else
  return 1.0 / x;
#endif
}
GP_HD double frsqrt(double x) {
#if defined(__CUDA_ARCH__)
  return rsqrt_nr(x);
#else
  return 1.0 / sqrt(x);
#endif
}
GP_HD void fsincos(double x, double *sn, double *cs) {
#if defined(__CUDA_ARCH__)
  sincos_fast(x, sn, cs);
#else
  *sn = sin(x);
  *cs = cos(x);
#endif
}

// FP32 forms for the single-precision variant (cfg.precision = 1).
GP_HD float frcp(float x) {
#if defined(__CUDA_ARCH__)
  // MUFU.RCP (about 1 ulp) + one Newton step, no denormal / slow-path branch (the integrator's finite
  // tests catch x = 0)
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return fmaf(y, fmaf(-x, y, 1.0f), y);
#else
  return 1.0f / x;
#endif
}
#if defined(__CUDACC__)
__device__ __noinline__ float2 sincosf_library(float x) {
  float2 r;
  sincosf(x, &r.x, &r.y);
  return r;   // by value, as sincos_library
}
// FP32 sincos for |x| < 1e4: two-term Cody-Waite (the FMA keeps q*hi exact), Taylor kernels through
// r^9 / r^10 on |r| <= pi/4 (truncation 2e-9 / 1e-10, below half an FP32 ulp), quadrant swap.
__device__ __forceinline__ void sincosf_fast(float x, float *sn, float *cs) {
  if (!(fabsf(x) < 1.0e4f)) {
    float2 sc = sincosf_library(x);
    *sn = sc.x;
    *cs = sc.y;
    return;
  }
  float qf = rintf(x * 0.636619772367581343f);
  int q = __float2int_rn(qf);
  float r = fmaf(-qf, 1.57079637050628662109375f, x);
  r = fmaf(-qf, -4.37113882867379116e-8f, r);
  float z = r * r;
  float ps = fmaf(z, 2.75573192e-6f, -1.98412698e-4f);
  float pc = fmaf(z, -2.75573192e-7f, 2.48015873e-5f);
  ps = fmaf(z, ps, 8.33333333e-3f);
  pc = fmaf(z, pc, -1.38888889e-3f);
  ps = fmaf(z, ps, -1.66666667e-1f);
  pc = fmaf(z, pc, 4.16666667e-2f);
  float sr = fmaf(r * z, ps, r);
  float cr = fmaf(z * z, pc, fmaf(-0.5f, z, 1.0f));
  float a = (q & 1) ? cr : sr;
  float b = (q & 1) ? sr : cr;
  *sn = (q & 2) ? -a : a;
  *cs = ((q + 1) & 2) ? -b : b;
}
#endif
GP_HD void fsincos(float x, float *sn, float *cs) {
#if defined(__CUDA_ARCH__)
  sincosf_fast(x, sn, cs);
#else
  *sn = sinf(x);
  *cs = cosf(x);
#endif
}
GP_HD float frsqrt(float x) {
#if defined(__CUDA_ARCH__)
  return rsqrtf(x);
#else
  return 1.0f / sqrtf(x);
#endif
}
GP_HD double fexp(double x) { return exp(x); }
GP_HD float fexp(float x) { return expf(x); }
GP_HD double fsqrt(double x) { return sqrt(x); }
GP_HD float fsqrt(float x) { return sqrtf(x); }
GP_HD double ffma(double a, double b, double c) { return fma(a, b, c); }
GP_HD float ffma(float a, float b, float c) { return fmaf(a, b, c); }

template <class T> struct identity_of { typedef T type; };

}  // namespace gp
#endif
