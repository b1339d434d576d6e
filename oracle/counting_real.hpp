// oracle/counting_real.hpp — TEST INFRASTRUCTURE. A double that tallies arithmetic, so that running the
// oracle text (mhm_oracle.hpp) with T = CountingReal yields the *algorithmic* FLOP count per cell-update
// of SURVEY.md §8(d). Convention: add = sub = mul = div = sqrt = min/max = 1 FLOP each;
// abs, negate, compare, select and copies = 0. The tally is what bench.py's roofline uses; it is
// recorded once in BASELINE.md / DESIGN.md and not tuned.
#pragma once
#include <cmath>

namespace mhm_oracle {

struct FlopTally {
  unsigned long long add = 0, mul = 0, div = 0, sqrt = 0, minmax = 0;
  unsigned long long total() const { return add + mul + div + sqrt + minmax; }
};

inline FlopTally& tally() {
  static thread_local FlopTally t;
  return t;
}

struct CountingReal {
  double v;
  CountingReal() : v(0.0) {}
  explicit CountingReal(double x) : v(x) {}
};

inline CountingReal operator+(CountingReal a, CountingReal b) { ++tally().add; return CountingReal(a.v + b.v); }
inline CountingReal operator-(CountingReal a, CountingReal b) { ++tally().add; return CountingReal(a.v - b.v); }
inline CountingReal operator*(CountingReal a, CountingReal b) { ++tally().mul; return CountingReal(a.v * b.v); }
inline CountingReal operator/(CountingReal a, CountingReal b) { ++tally().div; return CountingReal(a.v / b.v); }
inline CountingReal operator-(CountingReal a) { return CountingReal(-a.v); }
inline CountingReal o_sqrt(CountingReal x) { ++tally().sqrt; return CountingReal(std::sqrt(x.v)); }
inline CountingReal o_abs(CountingReal x) { return CountingReal(std::fabs(x.v)); }
inline CountingReal o_min(CountingReal a, CountingReal b) { ++tally().minmax; return a.v < b.v ? a : b; }
inline double o_value(CountingReal x) { return x.v; }

}  // namespace mhm_oracle
