// oracle/flop_scalar.h
//
// TEST INFRASTRUCTURE ONLY.  The counting scalar of oracle/flop_count*.cpp: + - * / sqrt pow = 1 flop each (the oracles have no
// FMA, so a*b+c = 2, matching FMA = 2 at peak); comparisons, abs, min/max, selects and negation = 0 flops (tallied separately).
#pragma once
#include <cmath>
#include <cstddef>

struct Tally { long long add, mul, div, sqrt_, pow_, cmp, abs_; };
static thread_local Tally g_tally = {0, 0, 0, 0, 0, 0, 0};

struct CR {
  double v;
  constexpr CR() : v(0) {}
  constexpr CR(double x) : v(x) {}
  explicit operator double() const { return v; }
};
inline CR operator+(CR a, CR b) { g_tally.add++; return CR(a.v + b.v); }
inline CR operator-(CR a, CR b) { g_tally.add++; return CR(a.v - b.v); }
inline CR operator*(CR a, CR b) { g_tally.mul++; return CR(a.v * b.v); }
inline CR operator/(CR a, CR b) { g_tally.div++; return CR(a.v / b.v); }
inline CR operator-(CR a) { return CR(-a.v); }
inline bool operator<(CR a, CR b) { g_tally.cmp++; return a.v < b.v; }
inline bool operator>(CR a, CR b) { g_tally.cmp++; return a.v > b.v; }
inline bool operator<=(CR a, CR b) { g_tally.cmp++; return a.v <= b.v; }
inline bool operator>=(CR a, CR b) { g_tally.cmp++; return a.v >= b.v; }
inline bool operator==(CR a, CR b) { g_tally.cmp++; return a.v == b.v; }
namespace std {
inline CR sqrt(CR a) { g_tally.sqrt_++; return CR(::sqrt(a.v)); }
inline CR fabs(CR a) { g_tally.abs_++; return CR(::fabs(a.v)); }
inline CR pow(CR a, CR b) { g_tally.pow_++; return CR(::pow(a.v, b.v)); }
}  // namespace std

