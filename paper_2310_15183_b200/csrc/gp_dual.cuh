// gp_dual.cuh — forward-mode dual numbers in two directions, used in-kernel for the
// Manko-Novikov metric derivatives (BASELINE.json north_star (b)).
//
// A Dual2 carries a value and its partial derivatives along two independent variables
// (here the prolate spheroidal x = (r-M)/k and y = cos(theta), eq 38-39).
// Everything is __host__ __device__ so that the launcher can evaluate the observer's metric
// on the host with plain doubles through the same templates.
#ifndef GP_DUAL_CUH_
#define GP_DUAL_CUH_

#include "gp_math.cuh"

namespace gp {

struct Dual2 {
  double v, dx, dy;
  GP_HD Dual2() {}
  GP_HD Dual2(double v_) : v(v_), dx(0.0), dy(0.0) {}
  GP_HD Dual2(double v_, double dx_, double dy_) : v(v_), dx(dx_), dy(dy_) {}
};

GP_HD Dual2 operator+(const Dual2 &a, const Dual2 &b) { return Dual2(a.v + b.v, a.dx + b.dx, a.dy + b.dy); }
GP_HD Dual2 operator-(const Dual2 &a, const Dual2 &b) { return Dual2(a.v - b.v, a.dx - b.dx, a.dy - b.dy); }
GP_HD Dual2 operator-(const Dual2 &a) { return Dual2(-a.v, -a.dx, -a.dy); }
GP_HD Dual2 operator+(const Dual2 &a, double b) { return Dual2(a.v + b, a.dx, a.dy); }
GP_HD Dual2 operator+(double b, const Dual2 &a) { return Dual2(a.v + b, a.dx, a.dy); }
GP_HD Dual2 operator-(const Dual2 &a, double b) { return Dual2(a.v - b, a.dx, a.dy); }
GP_HD Dual2 operator-(double b, const Dual2 &a) { return Dual2(b - a.v, -a.dx, -a.dy); }
GP_HD Dual2 operator*(const Dual2 &a, const Dual2 &b) {
  return Dual2(a.v * b.v, a.dx * b.v + a.v * b.dx, a.dy * b.v + a.v * b.dy);
}
GP_HD Dual2 operator*(const Dual2 &a, double b) { return Dual2(a.v * b, a.dx * b, a.dy * b); }
GP_HD Dual2 operator*(double b, const Dual2 &a) { return Dual2(a.v * b, a.dx * b, a.dy * b); }

// 1/a: one reciprocal, derivatives -a'/a^2
GP_HD Dual2 recip(const Dual2 &a) {
  double i = frcp(a.v);
  double m = -i * i;
  return Dual2(i, a.dx * m, a.dy * m);
}
GP_HD double recip(double a) { return frcp(a); }
GP_HD Dual2 operator/(const Dual2 &a, const Dual2 &b) { return a * recip(b); }
GP_HD Dual2 operator/(double a, const Dual2 &b) { return a * recip(b); }
GP_HD Dual2 operator/(const Dual2 &a, double b) { return a * frcp(b); }

GP_HD Dual2 dsqrt(const Dual2 &a) {
  double s = sqrt(a.v);
  double m = 0.5 * frcp(s);
  return Dual2(s, a.dx * m, a.dy * m);
}
GP_HD double dsqrt(double a) { return sqrt(a); }
GP_HD Dual2 dexp(const Dual2 &a) {
  double e = exp(a.v);
  return Dual2(e, a.dx * e, a.dy * e);
}
GP_HD double dexp(double a) { return exp(a); }
GP_HD Dual2 sqr(const Dual2 &a) {
  double t = 2.0 * a.v;
  return Dual2(a.v * a.v, t * a.dx, t * a.dy);
}
GP_HD double sqr(double a) { return a * a; }

GP_HD double value_of(const Dual2 &a) { return a.v; }
GP_HD double value_of(double a) { return a; }

}  // namespace gp
#endif
