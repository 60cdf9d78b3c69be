// TEST INFRASTRUCTURE — CPU oracle (see philox.hpp header).
//
// Forward-mode dual numbers with D tangents: the oracle's stand-in for the paper's
// "automatic differentiation" of the path contribution w.r.t. the primary-sample-space
// coordinates.  Every discrete decision is taken on the value
// part, i.e. frozen, exactly as AD would.  Also a tiny Vec3<T> usable with T = Real or
// T = Dual<Real, D>.
#pragma once
#include <cmath>

namespace orc {

template <class Real, int D> struct Dual {
  Real v;
  Real d[D];
  Dual() : v(0) { for (int i = 0; i < D; ++i) d[i] = 0; }
  Dual(Real c) : v(c) { for (int i = 0; i < D; ++i) d[i] = 0; }
  static Dual variable(Real c, int k) { Dual r(c); r.d[k] = Real(1); return r; }
};

#define ORC_DUAL_T template <class Real, int D>
#define ORC_DU Dual<Real, D>
ORC_DUAL_T inline ORC_DU operator-(const ORC_DU& a) { ORC_DU r; r.v = -a.v; for (int i = 0; i < D; ++i) r.d[i] = -a.d[i]; return r; }
ORC_DUAL_T inline ORC_DU operator+(const ORC_DU& a, const ORC_DU& b) { ORC_DU r; r.v = a.v + b.v; for (int i = 0; i < D; ++i) r.d[i] = a.d[i] + b.d[i]; return r; }
ORC_DUAL_T inline ORC_DU operator-(const ORC_DU& a, const ORC_DU& b) { ORC_DU r; r.v = a.v - b.v; for (int i = 0; i < D; ++i) r.d[i] = a.d[i] - b.d[i]; return r; }
ORC_DUAL_T inline ORC_DU operator*(const ORC_DU& a, const ORC_DU& b) { ORC_DU r; r.v = a.v * b.v; for (int i = 0; i < D; ++i) r.d[i] = a.d[i] * b.v + a.v * b.d[i]; return r; }
ORC_DUAL_T inline ORC_DU operator/(const ORC_DU& a, const ORC_DU& b) {
  ORC_DU r; const Real inv = Real(1) / b.v; r.v = a.v * inv;
  for (int i = 0; i < D; ++i) r.d[i] = (a.d[i] - r.v * b.d[i]) * inv;
  return r;
}
ORC_DUAL_T inline ORC_DU operator+(const ORC_DU& a, Real b) { ORC_DU r = a; r.v += b; return r; }
ORC_DUAL_T inline ORC_DU operator+(Real a, const ORC_DU& b) { return b + a; }
ORC_DUAL_T inline ORC_DU operator-(const ORC_DU& a, Real b) { ORC_DU r = a; r.v -= b; return r; }
ORC_DUAL_T inline ORC_DU operator-(Real a, const ORC_DU& b) { return (-b) + a; }
ORC_DUAL_T inline ORC_DU operator*(const ORC_DU& a, Real b) { ORC_DU r; r.v = a.v * b; for (int i = 0; i < D; ++i) r.d[i] = a.d[i] * b; return r; }
ORC_DUAL_T inline ORC_DU operator*(Real a, const ORC_DU& b) { return b * a; }
ORC_DUAL_T inline ORC_DU operator/(const ORC_DU& a, Real b) { return a * (Real(1) / b); }
ORC_DUAL_T inline ORC_DU operator/(Real a, const ORC_DU& b) { return ORC_DU(a) / b; }
ORC_DUAL_T inline ORC_DU& operator+=(ORC_DU& a, const ORC_DU& b) { a = a + b; return a; }
ORC_DUAL_T inline ORC_DU& operator*=(ORC_DU& a, const ORC_DU& b) { a = a * b; return a; }

// sqrt with the derivative set to 0 at 0 (the maps below reach 0 only on measure-zero sets).
ORC_DUAL_T inline ORC_DU sqrt(const ORC_DU& a) {
  ORC_DU r; r.v = std::sqrt(a.v);
  const Real k = a.v > Real(0) ? Real(0.5) / r.v : Real(0);
  for (int i = 0; i < D; ++i) r.d[i] = a.d[i] * k;
  return r;
}
ORC_DUAL_T inline ORC_DU sin(const ORC_DU& a) { ORC_DU r; r.v = std::sin(a.v); const Real c = std::cos(a.v); for (int i = 0; i < D; ++i) r.d[i] = a.d[i] * c; return r; }
ORC_DUAL_T inline ORC_DU cos(const ORC_DU& a) { ORC_DU r; r.v = std::cos(a.v); const Real s = -std::sin(a.v); for (int i = 0; i < D; ++i) r.d[i] = a.d[i] * s; return r; }
ORC_DUAL_T inline Real value(const ORC_DU& a) { return a.v; }
#undef ORC_DUAL_T
#undef ORC_DU

inline float value(float a) { return a; }
inline double value(double a) { return a; }
inline float sqrt(float a) { return std::sqrt(a); }
inline double sqrt(double a) { return std::sqrt(a); }
inline float sin(float a) { return std::sin(a); }
inline double sin(double a) { return std::sin(a); }
inline float cos(float a) { return std::cos(a); }
inline double cos(double a) { return std::cos(a); }

template <class T> struct Vec3 {
  T x, y, z;
  Vec3() : x(0), y(0), z(0) {}
  Vec3(T a, T b, T c) : x(a), y(b), z(c) {}
};
template <class T> inline Vec3<T> operator+(const Vec3<T>& a, const Vec3<T>& b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
template <class T> inline Vec3<T> operator-(const Vec3<T>& a, const Vec3<T>& b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
template <class T> inline Vec3<T> operator-(const Vec3<T>& a) { return {-a.x, -a.y, -a.z}; }
template <class T> inline Vec3<T> operator*(const Vec3<T>& a, const T& s) { return {a.x * s, a.y * s, a.z * s}; }
template <class T> inline T dot(const Vec3<T>& a, const Vec3<T>& b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <class T> inline Vec3<T> cross(const Vec3<T>& a, const Vec3<T>& b) {
  return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
template <class T> inline Vec3<T> normalize(const Vec3<T>& a) {
  using orc::sqrt;
  const T inv = T(1) / sqrt(dot(a, a));
  return a * inv;
}
// promote a constant Real vector to T
template <class T, class Real> inline Vec3<T> lift(const Vec3<Real>& a) { return {T(a.x), T(a.y), T(a.z)}; }

}  // namespace orc
