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

template <class S>
struct Dual2T {
  S v, dx, dy;
  GP_HD Dual2T() {}
  GP_HD Dual2T(S v_) : v(v_), dx(S(0)), dy(S(0)) {}
  GP_HD Dual2T(S v_, S dx_, S dy_) : v(v_), dx(dx_), dy(dy_) {}
};
typedef Dual2T<double> Dual2;

// plain scalars mixed with duals convert to the dual's scalar type (non-deduced parameter)
#define GP_S typename identity_of<S>::type

template <class S> GP_HD Dual2T<S> operator+(const Dual2T<S> &a, const Dual2T<S> &b) { return Dual2T<S>(a.v + b.v, a.dx + b.dx, a.dy + b.dy); }
template <class S> GP_HD Dual2T<S> operator-(const Dual2T<S> &a, const Dual2T<S> &b) { return Dual2T<S>(a.v - b.v, a.dx - b.dx, a.dy - b.dy); }
template <class S> GP_HD Dual2T<S> operator-(const Dual2T<S> &a) { return Dual2T<S>(-a.v, -a.dx, -a.dy); }
template <class S> GP_HD Dual2T<S> operator+(const Dual2T<S> &a, GP_S b) { return Dual2T<S>(a.v + b, a.dx, a.dy); }
template <class S> GP_HD Dual2T<S> operator+(GP_S b, const Dual2T<S> &a) { return Dual2T<S>(a.v + b, a.dx, a.dy); }
template <class S> GP_HD Dual2T<S> operator-(const Dual2T<S> &a, GP_S b) { return Dual2T<S>(a.v - b, a.dx, a.dy); }
template <class S> GP_HD Dual2T<S> operator-(GP_S b, const Dual2T<S> &a) { return Dual2T<S>(b - a.v, -a.dx, -a.dy); }
template <class S> GP_HD Dual2T<S> operator*(const Dual2T<S> &a, const Dual2T<S> &b) {
  return Dual2T<S>(a.v * b.v, a.dx * b.v + a.v * b.dx, a.dy * b.v + a.v * b.dy);
}
template <class S> GP_HD Dual2T<S> operator*(const Dual2T<S> &a, GP_S b) { return Dual2T<S>(a.v * b, a.dx * b, a.dy * b); }
template <class S> GP_HD Dual2T<S> operator*(GP_S b, const Dual2T<S> &a) { return Dual2T<S>(a.v * b, a.dx * b, a.dy * b); }

// 1/a: one reciprocal, derivatives -a'/a^2
template <class S> GP_HD Dual2T<S> recip(const Dual2T<S> &a) {
  S i = frcp(a.v);
  S m = -i * i;
  return Dual2T<S>(i, a.dx * m, a.dy * m);
}
GP_HD double recip(double a) { return frcp(a); }
GP_HD float recip(float a) { return frcp(a); }
template <class S> GP_HD Dual2T<S> operator/(const Dual2T<S> &a, const Dual2T<S> &b) { return a * recip(b); }
template <class S> GP_HD Dual2T<S> operator/(GP_S a, const Dual2T<S> &b) { return a * recip(b); }
template <class S> GP_HD Dual2T<S> operator/(const Dual2T<S> &a, GP_S b) { return a * frcp(b); }

template <class S> GP_HD Dual2T<S> dsqrt(const Dual2T<S> &a) {
  S s = fsqrt(a.v);
  S m = S(0.5) * frcp(s);
  return Dual2T<S>(s, a.dx * m, a.dy * m);
}
GP_HD double dsqrt(double a) { return sqrt(a); }
GP_HD float dsqrt(float a) { return sqrtf(a); }
// a^{-1/2}: one reciprocal square root, derivatives -a'/(2 a^{3/2})
template <class S> GP_HD Dual2T<S> drsqrt(const Dual2T<S> &a) {
  S i = frsqrt(a.v);
  S m = S(-0.5) * i * (i * i);
  return Dual2T<S>(i, a.dx * m, a.dy * m);
}
GP_HD double drsqrt(double a) { return frsqrt(a); }
GP_HD float drsqrt(float a) { return frsqrt(a); }
template <class S> GP_HD Dual2T<S> dexp(const Dual2T<S> &a) {
  S e = fexp(a.v);
  return Dual2T<S>(e, a.dx * e, a.dy * e);
}
GP_HD double dexp(double a) { return exp(a); }
GP_HD float dexp(float a) { return expf(a); }
template <class S> GP_HD Dual2T<S> sqr(const Dual2T<S> &a) {
  S t = S(2) * a.v;
  return Dual2T<S>(a.v * a.v, t * a.dx, t * a.dy);
}
GP_HD double sqr(double a) { return a * a; }
GP_HD float sqr(float a) { return a * a; }

template <class S> GP_HD S value_of(const Dual2T<S> &a) { return a.v; }
GP_HD double value_of(double a) { return a; }
#undef GP_S

}  // namespace gp
#endif
