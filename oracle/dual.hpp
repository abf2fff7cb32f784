// ORACLE — test infrastructure only (see oracle/README.md). Not part of the product path.
//
// Forward-mode tangent scalar: a value and ND directional derivatives carried through
// ordinary arithmetic.  Used by field.hpp to obtain the partial derivatives of the
// stationarity residual g(z; x*) of PAPER.md Eq. (2) (implicit-function form of the
// vector-field VJP).  30 lines of calculus rules, no library.
#pragma once
#include <cmath>

namespace orc {

constexpr int ND = 8;  // tangent directions propagated per pass

struct Dual {
  double v;
  double d[ND];
  Dual() : v(0.0) { for (int i = 0; i < ND; ++i) d[i] = 0.0; }
  Dual(double a) : v(a) { for (int i = 0; i < ND; ++i) d[i] = 0.0; }
};

inline double val(double a) { return a; }
inline double val(const Dual& a) { return a.v; }

inline Dual operator+(const Dual& a, const Dual& b) { Dual r; r.v = a.v + b.v; for (int i = 0; i < ND; ++i) r.d[i] = a.d[i] + b.d[i]; return r; }
inline Dual operator-(const Dual& a, const Dual& b) { Dual r; r.v = a.v - b.v; for (int i = 0; i < ND; ++i) r.d[i] = a.d[i] - b.d[i]; return r; }
inline Dual operator-(const Dual& a) { Dual r; r.v = -a.v; for (int i = 0; i < ND; ++i) r.d[i] = -a.d[i]; return r; }
inline Dual operator*(const Dual& a, const Dual& b) { Dual r; r.v = a.v * b.v; for (int i = 0; i < ND; ++i) r.d[i] = a.d[i] * b.v + a.v * b.d[i]; return r; }
inline Dual operator/(const Dual& a, const Dual& b) {
  Dual r; r.v = a.v / b.v;
  for (int i = 0; i < ND; ++i) r.d[i] = (a.d[i] - r.v * b.d[i]) / b.v;
  return r;
}
inline Dual& operator+=(Dual& a, const Dual& b) { a = a + b; return a; }
inline Dual& operator-=(Dual& a, const Dual& b) { a = a - b; return a; }
inline Dual& operator*=(Dual& a, const Dual& b) { a = a * b; return a; }

inline Dual chain(const Dual& a, double f, double df) { Dual r; r.v = f; for (int i = 0; i < ND; ++i) r.d[i] = df * a.d[i]; return r; }
inline Dual sqrt(const Dual& a) { double s = std::sqrt(a.v); return chain(a, s, 0.5 / s); }
inline Dual exp(const Dual& a) { double e = std::exp(a.v); return chain(a, e, e); }
inline Dual log(const Dual& a) { return chain(a, std::log(a.v), 1.0 / a.v); }
inline Dual sin(const Dual& a) { return chain(a, std::sin(a.v), std::cos(a.v)); }
inline Dual cos(const Dual& a) { return chain(a, std::cos(a.v), -std::sin(a.v)); }
// a^b for a > 0 (both may carry tangents); a == 0 handled by the caller.
inline Dual pow(const Dual& a, const Dual& b) {
  double f = std::pow(a.v, b.v);
  Dual r; r.v = f;
  double da = b.v * std::pow(a.v, b.v - 1.0), db = f * std::log(a.v);
  for (int i = 0; i < ND; ++i) r.d[i] = da * a.d[i] + db * b.d[i];
  return r;
}

using std::sqrt; using std::exp; using std::log; using std::sin; using std::cos; using std::pow;

}  // namespace orc
