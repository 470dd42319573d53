/* oracle/opcount.h — op-counting scalar for the oracle (TEST INFRASTRUCTURE / MEASUREMENT ONLY).
 *
 * With -DTFO_COUNT_OPS, tfo.cpp is compiled with `double` replaced by this class, which behaves like a double
 * and counts every FP64 operation the oracle's arithmetic performs ("exact counts from an op-counting
 * scalar type in the oracle").  The class has one double member, so the C ABI of tfo.h is unchanged in layout.
 * Counters are per thread: count with one OpenMP thread (tfo_set_num_threads(1)).  oracle/count_ops.py drives it. */
#ifndef TFO_OPCOUNT_H
#define TFO_OPCOUNT_H
#include <cmath>
#include <cstdint>

namespace tfo_count {
enum { ADD = 0, MUL = 1, DIV = 2, SQRT = 3, POW = 4, CMP = 5, ABSNEG = 6, N = 8 };
inline thread_local int64_t ops[N] = {0, 0, 0, 0, 0, 0, 0, 0};

struct real {
  double v;
  real() = default;
  real(double x) : v(x) {}
  real(int x) : v(x) {}
  real(long x) : v((double)x) {}
  real& operator+=(const real& o) { ++ops[ADD]; v += o.v; return *this; }
  real& operator-=(const real& o) { ++ops[ADD]; v -= o.v; return *this; }
  real& operator*=(const real& o) { ++ops[MUL]; v *= o.v; return *this; }
  real& operator/=(const real& o) { ++ops[DIV]; v /= o.v; return *this; }
  real operator-() const { ++ops[ABSNEG]; return real(-v); }
  real operator+() const { return *this; }
};
inline real operator+(const real& a, const real& b) { ++ops[ADD]; return real(a.v + b.v); }
inline real operator-(const real& a, const real& b) { ++ops[ADD]; return real(a.v - b.v); }
inline real operator*(const real& a, const real& b) { ++ops[MUL]; return real(a.v * b.v); }
inline real operator/(const real& a, const real& b) { ++ops[DIV]; return real(a.v / b.v); }
inline bool operator<(const real& a, const real& b) { ++ops[CMP]; return a.v < b.v; }
inline bool operator>(const real& a, const real& b) { ++ops[CMP]; return a.v > b.v; }
inline bool operator<=(const real& a, const real& b) { ++ops[CMP]; return a.v <= b.v; }
inline bool operator>=(const real& a, const real& b) { ++ops[CMP]; return a.v >= b.v; }
inline bool operator==(const real& a, const real& b) { ++ops[CMP]; return a.v == b.v; }
inline bool operator!=(const real& a, const real& b) { ++ops[CMP]; return a.v != b.v; }
inline bool operator!(const real& a) { return !a.v; }
}  // namespace tfo_count

namespace std {   /* the oracle calls these with the std:: prefix */
inline tfo_count::real sqrt(const tfo_count::real& a) { ++tfo_count::ops[tfo_count::SQRT]; return tfo_count::real(std::sqrt(a.v)); }
inline tfo_count::real fabs(const tfo_count::real& a) { ++tfo_count::ops[tfo_count::ABSNEG]; return tfo_count::real(std::fabs(a.v)); }
inline tfo_count::real pow(const tfo_count::real& a, const tfo_count::real& b) {
  ++tfo_count::ops[tfo_count::POW];
  return tfo_count::real(std::pow(a.v, b.v));
}
/* std::min / std::max with a literal on one side (the template cannot deduce one type for both) */
inline tfo_count::real min(double a, const tfo_count::real& b) { const tfo_count::real x(a); return b < x ? b : x; }
inline tfo_count::real min(const tfo_count::real& a, double b) { const tfo_count::real x(b); return x < a ? x : a; }
inline tfo_count::real max(double a, const tfo_count::real& b) { const tfo_count::real x(a); return x < b ? b : x; }
inline tfo_count::real max(const tfo_count::real& a, double b) { const tfo_count::real x(b); return a < x ? x : a; }
}  // namespace std
#endif
