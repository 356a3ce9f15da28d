// ORACLE — TEST INFRASTRUCTURE ONLY.  Nothing under oracle/ is part of the product path.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may use it.
//
// real.hpp: the scalar types the oracle is templated on (double = the oracle proper,
// long double and __float128 = referees for disagreements at the 1e-10 level, Counted = an
// operation-counting double used to state the algorithmic flop count),
// elementary-function overloads for each, and a minimal complex number.
#pragma once
#include <cmath>
#include <cstdint>
#include <quadmath.h>

namespace mfo {

// ---- elementary functions, one overload per real type -------------------------------------
inline double r_sqrt(double x) { return std::sqrt(x); }
inline double r_log(double x) { return std::log(x); }
inline double r_exp(double x) { return std::exp(x); }
inline double r_sin(double x) { return std::sin(x); }
inline double r_cos(double x) { return std::cos(x); }
inline double r_atan2(double y, double x) { return std::atan2(y, x); }
inline double r_asinh(double x) { return std::asinh(x); }
inline double r_pow(double x, double y) { return std::pow(x, y); }
inline double r_fabs(double x) { return std::fabs(x); }
inline double r_to_double(double x) { return x; }

inline long double r_sqrt(long double x) { return sqrtl(x); }
inline long double r_log(long double x) { return logl(x); }
inline long double r_exp(long double x) { return expl(x); }
inline long double r_sin(long double x) { return sinl(x); }
inline long double r_cos(long double x) { return cosl(x); }
inline long double r_atan2(long double y, long double x) { return atan2l(y, x); }
inline long double r_asinh(long double x) { return asinhl(x); }
inline long double r_pow(long double x, long double y) { return powl(x, y); }
inline long double r_fabs(long double x) { return fabsl(x); }
inline double r_to_double(long double x) { return (double)x; }

inline __float128 r_sqrt(__float128 x) { return sqrtq(x); }
inline __float128 r_log(__float128 x) { return logq(x); }
inline __float128 r_exp(__float128 x) { return expq(x); }
inline __float128 r_sin(__float128 x) { return sinq(x); }
inline __float128 r_cos(__float128 x) { return cosq(x); }
inline __float128 r_atan2(__float128 y, __float128 x) { return atan2q(y, x); }
inline __float128 r_asinh(__float128 x) { return asinhq(x); }
inline __float128 r_pow(__float128 x, __float128 y) { return powq(x, y); }
inline __float128 r_fabs(__float128 x) { return fabsq(x); }
inline double r_to_double(__float128 x) { return (double)x; }

// ---- operation-counting double ------------------------------------------------------------
struct OpCounts {
  uint64_t add = 0, mul = 0, div = 0, sqrt = 0, trans = 0, cmp = 0;
};
inline OpCounts& op_counts() {
  static OpCounts c;
  return c;
}
struct Counted {
  double v;
  Counted() : v(0) {}
  Counted(double x) : v(x) {}
  Counted(int x) : v(x) {}
  explicit Counted(long double x) : v((double)x) {}
  explicit Counted(__float128 x) : v((double)x) {}
  explicit operator double() const { return v; }
  explicit operator long double() const { return v; }
  explicit operator int() const { return (int)v; }
};
inline Counted operator+(Counted a, Counted b) { op_counts().add++; return Counted(a.v + b.v); }
inline Counted operator-(Counted a, Counted b) { op_counts().add++; return Counted(a.v - b.v); }
inline Counted operator*(Counted a, Counted b) { op_counts().mul++; return Counted(a.v * b.v); }
inline Counted operator/(Counted a, Counted b) { op_counts().div++; return Counted(a.v / b.v); }
inline Counted operator-(Counted a) { return Counted(-a.v); }
inline Counted& operator+=(Counted& a, Counted b) { a = a + b; return a; }
inline Counted& operator-=(Counted& a, Counted b) { a = a - b; return a; }
inline Counted& operator*=(Counted& a, Counted b) { a = a * b; return a; }
inline Counted& operator/=(Counted& a, Counted b) { a = a / b; return a; }
inline bool operator<(Counted a, Counted b) { op_counts().cmp++; return a.v < b.v; }
inline bool operator>(Counted a, Counted b) { op_counts().cmp++; return a.v > b.v; }
inline bool operator<=(Counted a, Counted b) { op_counts().cmp++; return a.v <= b.v; }
inline bool operator>=(Counted a, Counted b) { op_counts().cmp++; return a.v >= b.v; }
inline bool operator==(Counted a, Counted b) { op_counts().cmp++; return a.v == b.v; }
inline bool operator!=(Counted a, Counted b) { op_counts().cmp++; return a.v != b.v; }
inline Counted r_sqrt(Counted x) { op_counts().sqrt++; return Counted(std::sqrt(x.v)); }
inline Counted r_log(Counted x) { op_counts().trans++; return Counted(std::log(x.v)); }
inline Counted r_exp(Counted x) { op_counts().trans++; return Counted(std::exp(x.v)); }
inline Counted r_sin(Counted x) { op_counts().trans++; return Counted(std::sin(x.v)); }
inline Counted r_cos(Counted x) { op_counts().trans++; return Counted(std::cos(x.v)); }
inline Counted r_atan2(Counted y, Counted x) { op_counts().trans++; return Counted(std::atan2(y.v, x.v)); }
inline Counted r_asinh(Counted x) { op_counts().trans++; return Counted(std::asinh(x.v)); }
inline Counted r_pow(Counted x, Counted y) { op_counts().trans++; return Counted(std::pow(x.v, y.v)); }
inline Counted r_fabs(Counted x) { return Counted(std::fabs(x.v)); }
inline double r_to_double(Counted x) { return x.v; }

// ---- constants ----------------------------------------------------------------------------
template <class R> inline R r_pi() { return R(3.14159265358979323846264338327950288419716939937510582Q); }

// ---- minimal complex number (no library complex: keeps every operation visible) ------------
template <class R> struct Cx {
  R re, im;
  Cx() : re(R(0)), im(R(0)) {}
  Cx(R r) : re(r), im(R(0)) {}
  Cx(R r, R i) : re(r), im(i) {}
};
template <class R> inline Cx<R> operator+(Cx<R> a, Cx<R> b) { return Cx<R>(a.re + b.re, a.im + b.im); }
template <class R> inline Cx<R> operator-(Cx<R> a, Cx<R> b) { return Cx<R>(a.re - b.re, a.im - b.im); }
template <class R> inline Cx<R> operator-(Cx<R> a) { return Cx<R>(-a.re, -a.im); }
template <class R> inline Cx<R> operator*(Cx<R> a, Cx<R> b) {
  return Cx<R>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <class R> inline Cx<R> operator*(R s, Cx<R> a) { return Cx<R>(s * a.re, s * a.im); }
template <class R> inline Cx<R> operator*(Cx<R> a, R s) { return Cx<R>(s * a.re, s * a.im); }
template <class R> inline Cx<R> operator/(Cx<R> a, R s) { return Cx<R>(a.re / s, a.im / s); }
template <class R> inline Cx<R>& operator+=(Cx<R>& a, Cx<R> b) { a = a + b; return a; }
template <class R> inline Cx<R> conj(Cx<R> a) { return Cx<R>(a.re, -a.im); }
template <class R> inline R norm2(Cx<R> a) { return a.re * a.re + a.im * a.im; }
template <class R> inline Cx<R> cx_i() { return Cx<R>(R(0), R(1)); }

}  // namespace mfo
