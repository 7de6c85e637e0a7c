// oracle/flop_count.cpp
//
// TEST INFRASTRUCTURE ONLY (see hydro_oracle.cpp).  Instantiates the oracle's templates with a
// counting scalar to obtain the ALGORITHMIC operation count of one patch-group update as the oracle
// states it (SURVEY.md 8(d) "Algorithmic flop count, exactly"):  + - * / sqrt pow = 1 flop each (the
// oracle has no FMA, so a*b+c = 2, matching FMA = 2 at peak); comparisons, abs, min/max, selects and
// negation = 0 flops (tallied separately).  Data-dependent work (limiter zero branch, HLLC branch,
// Newton iterations) is whatever the given input takes.  Used by oracle/count_flops.py only.
#include "flop_scalar.h"

#include "hydro_oracle.cpp"

namespace {
template <> struct ExactTol<CR> { static constexpr double v = 1e-12; };
}  // namespace

extern "C" {
// counts[8]: add, mul, div, sqrt, pow, cmp, abs, riemann solves; summed over the Ng groups of `in` (fp64 input)
int oracle_count_ops(const double* in, int Ng, int g, double dt, double dh, double gamma, int scheme, int riemann_, int limiter,
                     int recon, int char_limit, int want_flux, long long* counts) {
  Params<CR> p;
  p.gamma = gamma;
  p.nu = dt / dh;
  p.scheme = scheme;
  p.riemann = riemann_;
  p.limiter = limiter;
  p.recon = recon;
  p.char_limit = char_limit;
  p.roe_fallback = 1;
  p.theta = 1.5;
  p.min_dens = 0;
  p.min_pres = 0;
  const int S = PS + 2 * g;
  const size_t nin = (size_t)5 * S * S * S;
  std::vector<CR> cin(nin), cout((size_t)5 * PS * PS * PS), cff((size_t)9 * 5 * PS * PS);
  g_tally = {0, 0, 0, 0, 0, 0, 0};
  Status st;
  for (int gi = 0; gi < Ng; ++gi) {
    for (size_t x = 0; x < nin; ++x) cin[x] = CR(in[gi * nin + x]);
    solve_group<CR>(cin.data(), cout.data(), want_flux ? cff.data() : nullptr, g, p, &st);
  }
  counts[0] = g_tally.add; counts[1] = g_tally.mul; counts[2] = g_tally.div; counts[3] = g_tally.sqrt_;
  counts[4] = g_tally.pow_; counts[5] = g_tally.cmp; counts[6] = g_tally.abs_; counts[7] = st.c[3];
  return 0;
}
}
