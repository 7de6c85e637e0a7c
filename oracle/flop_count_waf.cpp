// oracle/flop_count_waf.cpp
//
// TEST INFRASTRUCTURE ONLY (see waf_oracle.cpp).  The split weighted-average-flux oracle instantiated with the counting scalar of
// flop_scalar.h: the ALGORITHMIC operation count of one patch-group update (three sweeps over the ranges the oracle sweeps) as
// the oracle states it.  Used by oracle/count_flops.py only.
#include "flop_scalar.h"

#include "waf_oracle.cpp"

extern "C" {
// counts[7]: add, mul, div, sqrt, pow, cmp, abs; summed over the Ng groups of `in` (fp64 input)
int oracle_waf_count_ops(const double* in, int Ng, int g, double dt, double dh, double gamma, int order, long long* counts) {
  const int S = PS + 2 * g;
  const size_t nin = (size_t)5 * S * S * S;
  std::vector<CR> cin(nin), cout((size_t)5 * PS * PS * PS), cff((size_t)9 * 5 * PS * PS);
  g_tally = {0, 0, 0, 0, 0, 0, 0};
  long long st[2] = {0, 0};
  for (int gi = 0; gi < Ng; ++gi) {
    for (size_t x = 0; x < nin; ++x) cin[x] = CR(in[gi * nin + x]);
    solve_group<CR>(cin.data(), cout.data(), cff.data(), g, CR(dt / dh), CR(gamma), order, st);
  }
  counts[0] = g_tally.add; counts[1] = g_tally.mul; counts[2] = g_tally.div; counts[3] = g_tally.sqrt_;
  counts[4] = g_tally.pow_; counts[5] = g_tally.cmp; counts[6] = g_tally.abs_;
  return 0;
}
}
