// mvwsa.h -- CPU side of MV-WSA (§3.3-3.5, Eq. 2-5; App. B Eq. 6-8).
// Plain host C++; no CUDA.  Readings G10/G11 of DESIGN.md.
#pragma once
#include <cmath>
#include <cstdint>
#include <vector>

namespace wisp {
namespace mvwsa {

struct Split { int64_t C; int64_t kappa; bool moved; };

// Eq. 6-8: kappa~ = max(kappa_min, ceil((1+h)p)); C~ = clip(floor((B - kappa~ b)/a), C_min, C_max);
// kappa~ <- floor((B - C~ a)/b); dead zone Delta.
inline Split live_law(uint64_t B, uint64_t a, uint64_t b, uint64_t kappa_floor, double p, double h, int64_t c_min,
                      int64_t c_max, int64_t c_cur, int64_t delta) {
  const double want = std::ceil((1.0 + h) * p);
  uint64_t k1 = want > (double)kappa_floor ? (uint64_t)want : kappa_floor;
  int64_t ct = (k1 * b > B) ? 0 : (int64_t)((B - k1 * b) / a);
  if (ct < c_min) ct = c_min;
  if (ct > c_max) ct = c_max;
  if (std::llabs(ct - c_cur) < delta) return {c_cur, (int64_t)((B - (uint64_t)c_cur * a) / b), false};
  return {ct, (int64_t)((B - (uint64_t)ct * a) / b), true};
}

// m(C) = sum_{dist > C} hist[dist]; hist has E+2 bins, bin E+1 = infinite distance.
inline std::vector<double> miss_curve(const std::vector<double>& hist, int E) {
  std::vector<double> m(E + 1);
  double tot = 0;
  for (int dd = 1; dd <= E + 1; ++dd) tot += hist[dd];
  double acc = 0;
  for (int C = 0; C <= E; ++C) {
    if (C >= 1) acc += hist[C];
    m[C] = tot - acc;
  }
  return m;
}

// G11: C_max = smallest C with m(C) == m(E) (beyond the knee extra slots are worth nothing).
inline int knee(const std::vector<double>& m, int E) {
  int c = E;
  while (c > 1 && m[c - 1] <= m[E]) --c;
  return c;
}

// Eq. 2-5: argmin over C in [c_min, min(c_max, C_feas)] of c_exp*m_exp(C) + c_kv*m_kv(kappa(C)); ties ->
// smaller C.  Returns -1 when the range is empty.
inline int64_t configurator(uint64_t B, uint64_t a, uint64_t b, uint64_t kappa_floor, double c_exp, double c_kv,
                            const std::vector<double>& m_exp, const double* m_kv, uint64_t m_kv_len, int64_t c_min,
                            int64_t c_max) {
  if (kappa_floor * b > B) return -1;
  const int64_t c_feas = (int64_t)((B - kappa_floor * b) / a);
  const int64_t hi = c_max < c_feas ? c_max : c_feas;
  int64_t best = -1;
  double best_t = 0;
  for (int64_t C = c_min; C <= hi; ++C) {
    const uint64_t kap = (B - (uint64_t)C * a) / b;
    double mk = 0;
    if (m_kv && m_kv_len) mk = m_kv[kap < m_kv_len ? kap : m_kv_len - 1];
    const double t = c_exp * m_exp[(size_t)C < m_exp.size() ? C : m_exp.size() - 1] + c_kv * mk;
    if (best < 0 || t < best_t) { best = C; best_t = t; }
  }
  return best;
}

}  // namespace mvwsa
}  // namespace wisp
