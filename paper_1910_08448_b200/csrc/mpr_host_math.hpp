// mpr_host_math.hpp -- host-only numerics of libmpr.so: the binned standard error of an energy
// series (R16) and the temperature-matching root search (R6, steps 1-5).
// Written from the text of those two readings; no CUDA in here, so that both pieces can be
// driven with synthetic inputs through mpr_debug_series_stats / mpr_debug_match_temperature and
// pinned against hand-worked numbers without a GPU (tests/test_host_logic.py).
#pragma once
#include <cmath>
#include <cstddef>
#include <limits>

namespace mpr_host {

// R16.  n samples -> (mean over all n, standard error).  B = 10 blocks when n >= 20, otherwise
// every sample is its own block; block length m = floor(n / B); samples past B m enter the
// mean but no block.  s.e. = sqrt( unbiased variance of the B block means / B ).
// Block means are folded into a running (mean, M2) pair as they complete (Welford), so no
// scratch array is needed.
struct SeriesStats {
  double mean = std::numeric_limits<double>::quiet_NaN();
  double stderr_ = 0.0;
};

inline SeriesStats series_stats(const double* e, std::size_t n) {
  SeriesStats r;
  if (n == 0) return r;
  long double total = 0.0L;
  for (std::size_t i = 0; i < n; ++i) total += e[i];
  r.mean = static_cast<double>(total / static_cast<long double>(n));
  if (n < 2) return r;
  const std::size_t blocks = n >= 20 ? 10 : n;
  const std::size_t m = n / blocks;
  double run_mean = 0.0, run_m2 = 0.0;
  const double* p = e;
  for (std::size_t b = 1; b <= blocks; ++b, p += m) {
    double s = 0.0;
    for (std::size_t i = 0; i < m; ++i) s += p[i];
    const double bm = s / static_cast<double>(m);
    const double d = bm - run_mean;
    run_mean += d / static_cast<double>(b);
    run_m2 += d * (bm - run_mean);
  }
  const double var = run_m2 / static_cast<double>(blocks - 1);
  r.stderr_ = std::sqrt(var / static_cast<double>(blocks));
  return r;
}

// R6.  The search is a small state machine so that the caller (which owns the GPU chain) stays
// in charge of running the trials:   while (m.want_trial()) m.report(gap(m.T()), se);
// gap = e_trial(T) - e_sample.  A bracket end is a (T, g) pair; `cold` has g <= 0, `warm` g >= 0.
class TemperatureMatcher {
 public:
  enum Outcome { SEARCHING, FOUND, NO_ROOT_BELOW, NO_ROOT_ABOVE };

  bool want_trial() const { return outcome_ == SEARCHING; }
  double T() const { return next_T_; }
  Outcome outcome() const { return outcome_; }
  double result() const { return answer_; }
  int trials() const { return trials_; }

  void report(double gap, double se) {
    ++trials_;
    switch (phase_) {
      case FIRST:            // step 1: the trial at T = 1e-4
        if (gap > 0.0) {     // step 2: already warmer than the sample -> walk down by decades
          warm_ = End{next_T_, gap};
          descend();
        } else {             // step 3: look at T = 1
          cold_ = End{next_T_, gap};
          phase_ = UP;
          next_T_ = kTopStart;
        }
        break;
      case DOWN:
        if (gap > 0.0) {
          warm_ = End{next_T_, gap};
          descend();
        } else {
          cold_ = End{next_T_, gap};
          begin_refine();
        }
        break;
      case UP:
        if (gap < 0.0) {
          if (next_T_ >= kCeiling) { outcome_ = NO_ROOT_ABOVE; break; }
          cold_ = End{next_T_, gap};
          next_T_ *= 10.0;
        } else {
          warm_ = End{next_T_, gap};
          begin_refine();
        }
        break;
      case REFINE: {         // step 4
        const double Tc = next_T_;
        answer_ = Tc;
        if (std::fabs(gap) <= 2.0 * se) { outcome_ = FOUND; break; }
        const int side = gap < 0.0 ? -1 : +1;
        if (side < 0) {
          cold_ = End{Tc, gap};
          if (prev_side_ < 0) warm_.g *= 0.5;      // Illinois: same end twice -> down-weight the other
        } else {
          warm_ = End{Tc, gap};
          if (prev_side_ > 0) cold_.g *= 0.5;
        }
        prev_side_ = side;
        const bool settled = refine_steps_ > 1 && std::fabs(Tc - prev_Tc_) / Tc < 0.01;
        prev_Tc_ = Tc;
        if (settled || refine_steps_ >= kMaxRefine) { outcome_ = FOUND; break; }
        propose();
        break;
      }
    }
  }

 private:
  struct End { double T, g; };
  enum Phase { FIRST, DOWN, UP, REFINE };
  static constexpr double kBottomStart = 1e-4, kTopStart = 1.0;
  static constexpr double kFloor = 1.5e-6, kCeiling = 0.99e2;   // 1e-6 and 1e2 are the last decades tried
  static constexpr int kMaxRefine = 20;

  void descend() {
    if (next_T_ <= kFloor) { outcome_ = NO_ROOT_BELOW; return; }
    phase_ = DOWN;
    next_T_ = next_T_ / 10.0;
  }
  void begin_refine() {
    phase_ = REFINE;
    answer_ = warm_.T;
    prev_Tc_ = warm_.T;
    propose();
  }
  void propose() {   // secant through the two ends; midpoint when it leaves the open bracket
    ++refine_steps_;
    double Tc = warm_.T - warm_.g * (warm_.T - cold_.T) / (warm_.g - cold_.g);
    if (!(Tc > cold_.T && Tc < warm_.T)) Tc = 0.5 * (cold_.T + warm_.T);
    next_T_ = Tc;
  }

  Phase phase_ = FIRST;
  Outcome outcome_ = SEARCHING;
  End cold_{0.0, 0.0}, warm_{0.0, 0.0};
  double next_T_ = kBottomStart, answer_ = 0.0, prev_Tc_ = 0.0;
  int prev_side_ = 0, refine_steps_ = 0, trials_ = 0;
};

}  // namespace mpr_host
