// jitter_trig.h — TEST SUPPORT for the oracle-only rounding experiment (SURVEY.md App. B-6 style).
// Force-included (-include) into a second build of oracle/aw_oracle.cpp, whose source stays untouched: every
// std::sin / std::cos result is moved by -1, 0 or +1 ulp, chosen by a hash of the argument's bits.  This is the
// size of the difference between two correct sincos implementations (libm vs any <= 1-ulp routine), so the
// spread it causes in an output (dH_max, FLI, class) is rounding noise no parity bar may be tighter than.
#pragma once
#include <cmath>
#include <cstdint>
#include <cstring>
namespace std {
inline double aw_jitter(double x, double v, uint64_t salt) {
  uint64_t b;
  std::memcpy(&b, &x, 8);
  b = (b ^ salt) * 0x9E3779B97F4A7C15ull;
  b ^= b >> 29;
  b *= 0xBF58476D1CE4E5B9ull;
  b ^= b >> 32;
  const unsigned r = (unsigned)(b % 3u);
  if (r == 0 || v == 0.0 || !(v == v)) return v;
  return std::nextafter(v, r == 1 ? 2.0 : -2.0);
}
inline double aw_jitter_sin(double x) { return aw_jitter(x, sin(x), 0x1234567ull); }
inline double aw_jitter_cos(double x) { return aw_jitter(x, cos(x), 0x7654321ull); }
}  // namespace std
#define sin aw_jitter_sin
#define cos aw_jitter_cos
