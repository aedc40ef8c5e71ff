// Closed-form SU(2) recoupling coefficients for the host symmetry layer (F-5).
// Racah's formula for the 6j symbol in long double, the 9j symbol as a sum over 6j products.
// All angular momenta are passed doubled (tj = 2j).  On the hot path s, s', k, r, k' are 0 or
// 1/2, so every sum has at most a few terms and no cancellation to speak of.
#include <cmath>
#include <unordered_map>

#include "fh_internal.hpp"

#include <stdexcept>

namespace fh {

// n! as long double, n < FACT_MAX (labels with 2j up to ~250; mps_set_bond / mps_load refuse larger ones).
// The table is built by a function-local static initialiser: thread safe (the two-site plans are emitted on a
// second host thread).
static const int FACT_MAX = 800;
struct FactTable {
  long double v[FACT_MAX];
  FactTable() {
    v[0] = 1.0L;
    for (int i = 1; i < FACT_MAX; ++i) v[i] = v[i - 1] * (long double)i;
  }
};
static long double fact(int n) {
  static const FactTable table;
  if (n < 0 || n >= FACT_MAX) throw std::out_of_range("recoupling coefficient: label out of the supported range");
  return table.v[n];
}

// Delta(a,b,c)^2 with doubled arguments
static long double delta2(int ta, int tb, int tc) {
  return fact((ta + tb - tc) / 2) * fact((ta - tb + tc) / 2) * fact((-ta + tb + tc) / 2) /
         fact((ta + tb + tc) / 2 + 1);
}

double wigner6j(int ta, int tb, int tc, int td, int te, int tf) {
  if (!triangle(ta, tb, tc) || !triangle(ta, te, tf) || !triangle(td, tb, tf) || !triangle(td, te, tc))
    return 0.0;
  const int a1 = (ta + tb + tc) / 2, a2 = (ta + te + tf) / 2, a3 = (td + tb + tf) / 2, a4 = (td + te + tc) / 2;
  const int b1 = (ta + tb + td + te) / 2, b2 = (tb + tc + te + tf) / 2, b3 = (tc + ta + tf + td) / 2;
  int tmin = a1;
  if (a2 > tmin) tmin = a2;
  if (a3 > tmin) tmin = a3;
  if (a4 > tmin) tmin = a4;
  int tmax = b1;
  if (b2 < tmax) tmax = b2;
  if (b3 < tmax) tmax = b3;
  long double sum = 0.0L;
  for (int t = tmin; t <= tmax; ++t) {
    long double term = fact(t + 1) / (fact(t - a1) * fact(t - a2) * fact(t - a3) * fact(t - a4) *
                                      fact(b1 - t) * fact(b2 - t) * fact(b3 - t));
    sum += (t & 1) ? -term : term;
  }
  long double pref = sqrtl(delta2(ta, tb, tc) * delta2(ta, te, tf) * delta2(td, tb, tf) * delta2(td, te, tc));
  return (double)(pref * sum);
}

// {j1 j2 j3; j4 j5 j6; j7 j8 j9} = sum_x (-1)^{2x} (2x+1) {j1 j4 j7; j8 j9 x} {j2 j5 j8; j4 x j6} {j3 j6 j9; x j1 j2}
static double wigner9j_sum(int j1, int j2, int j3, int j4, int j5, int j6, int j7, int j8, int j9);

// A plan asks for the same few hundred symbols tens of thousands of times (one per task): memoised per
// thread on the nine doubled arguments (7 bits each); the stored value is the one the sum returns.
double wigner9j(int j1, int j2, int j3, int j4, int j5, int j6, int j7, int j8, int j9) {
  const int a[9] = {j1, j2, j3, j4, j5, j6, j7, j8, j9};
  uint64_t key = 0;
  bool packable = true;
  for (int i = 0; i < 9; ++i) {
    packable = packable && a[i] >= 0 && a[i] < 128;
    key = (key << 7) | (uint64_t)(a[i] & 127);
  }
  if (!packable) return wigner9j_sum(j1, j2, j3, j4, j5, j6, j7, j8, j9);
  thread_local std::unordered_map<uint64_t, double> memo;
  auto it = memo.find(key);
  if (it != memo.end()) return it->second;
  const double v = wigner9j_sum(j1, j2, j3, j4, j5, j6, j7, j8, j9);
  if (memo.size() < (1u << 20)) memo.emplace(key, v);
  return v;
}

static double wigner9j_sum(int j1, int j2, int j3, int j4, int j5, int j6, int j7, int j8, int j9) {
  if (!triangle(j1, j2, j3) || !triangle(j4, j5, j6) || !triangle(j7, j8, j9) || !triangle(j1, j4, j7) ||
      !triangle(j2, j5, j8) || !triangle(j3, j6, j9))
    return 0.0;
  int lo = std::abs(j1 - j9);
  if (std::abs(j4 - j8) > lo) lo = std::abs(j4 - j8);
  if (std::abs(j2 - j6) > lo) lo = std::abs(j2 - j6);
  int hi = j1 + j9;
  if (j4 + j8 < hi) hi = j4 + j8;
  if (j2 + j6 < hi) hi = j2 + j6;
  long double sum = 0.0L;
  for (int tx = lo; tx <= hi; tx += 2) {
    long double term = (long double)(tx + 1) * (long double)wigner6j(j1, j4, j7, j8, j9, tx) *
                       (long double)wigner6j(j2, j5, j8, j4, tx, j6) * (long double)wigner6j(j3, j6, j9, tx, j1, j2);
    sum += (tx & 1) ? -term : term;
  }
  return (double)sum;
}

// coefL(a,s,c; k,r,k'; a',s',c') = sqrt((2c+1)(2k'+1)(2a'+1)(2s'+1)) {a s c; k r k'; a' s' c'}
double coef_left(int ta, int ts, int tc, int tk, int tr, int tkp, int tap, int tsp, int tcp) {
  const double nj = wigner9j(ta, ts, tc, tk, tr, tkp, tap, tsp, tcp);
  if (nj == 0.0) return 0.0;
  return std::sqrt((double)((tc + 1) * (tkp + 1) * (tap + 1) * (tsp + 1))) * nj;
}

// coefR(c,s,b; k,r,k'; c',s',b') = (2b'+1)/(2c'+1) sqrt((2b+1)(2k'+1)(2c'+1)(2s'+1)) {c s b; k r k'; c' s' b'}
double coef_right(int tc, int ts, int tb, int tk, int tr, int tkp, int tcp, int tsp, int tbp) {
  const double nj = wigner9j(tc, ts, tb, tk, tr, tkp, tcp, tsp, tbp);
  if (nj == 0.0) return 0.0;
  return (double)(tbp + 1) / (double)(tcp + 1) *
         std::sqrt((double)((tb + 1) * (tkp + 1) * (tcp + 1) * (tsp + 1))) * nj;
}

}  // namespace fh
