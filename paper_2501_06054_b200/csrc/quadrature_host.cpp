#include "quadrature_host.h"

#include <cstdint>
#include <cstring>
#include <map>
#include <mutex>

#include <algorithm>
#include <cmath>
#include <limits>

namespace sas {

// Number of eigenvalues of the Jacobi matrix that are < x (Sturm sequence of the LDL^T pivots).
static int sturm_count(const std::vector<double>& a, const std::vector<double>& b2, double x) {
  const double tiny = std::numeric_limits<double>::min();
  int cnt = 0;
  double d = 1.0;
  for (size_t k = 0; k < a.size(); ++k) {
    double off = (k == 0) ? 0.0 : b2[k] / d;
    d = (a[k] - x) - off;
    if (d == 0.0) d = -tiny;
    if (d < 0.0) ++cnt;
  }
  return cnt;
}

void gauss_from_jacobi(const std::vector<double>& a, const std::vector<double>& b, std::vector<double>& x,
                       std::vector<double>& w) {
  const int n = (int)a.size();
  x.assign(n, 0.0);
  w.assign(n, 0.0);
  std::vector<double> b2(n, 0.0);
  for (int k = 1; k < n; ++k) b2[k] = b[k] * b[k];
  // Gershgorin bounds
  double lo = a[0], hi = a[0];
  for (int k = 0; k < n; ++k) {
    double r = (k > 0 ? std::fabs(b[k]) : 0.0) + (k + 1 < n ? std::fabs(b[k + 1]) : 0.0);
    lo = std::min(lo, a[k] - r);
    hi = std::max(hi, a[k] + r);
  }
  for (int i = 0; i < n; ++i) {
    // eigenvalue i (ascending): smallest x with count(x) >= i+1
    double l = lo, h = hi;
    for (int it = 0; it < 200; ++it) {
      double m = 0.5 * (l + h);
      if (m <= l || m >= h) break;
      if (sturm_count(a, b2, m) >= i + 1) h = m; else l = m;
    }
    x[i] = 0.5 * (l + h);
  }
  // Christoffel numbers: w_i = 1 / sum_k p_k(x_i)^2 with orthonormal p_k, p_0 = 1.
  double wsum = 0.0;
  for (int i = 0; i < n; ++i) {
    double pm = 0.0, p = 1.0, s = 1.0;
    for (int k = 0; k + 1 < n; ++k) {
      double pn = ((x[i] - a[k]) * p - (k > 0 ? b[k] : 0.0) * pm) / b[k + 1];
      pm = p;
      p = pn;
      s += p * p;
    }
    w[i] = 1.0 / s;
    wsum += w[i];
  }
  for (int i = 0; i < n; ++i) w[i] /= wsum;
}

static void schulz_rule_compute(double p, int n, std::vector<double>& s, std::vector<double>& w) {
  if (n <= 1 || !(p > 0.0)) {
    s.assign(1, 1.0);
    w.assign(1, 1.0);
    return;
  }
  // f(r) ~ r^z exp(-(z+1) r / mean): generalised Laguerre weight x^alpha e^-x with alpha = z
  const double z = 1.0 / (p * p) - 1.0;
  std::vector<double> a(n), b(n, 0.0);
  for (int k = 0; k < n; ++k) {
    a[k] = 2.0 * k + 1.0 + z;
    if (k > 0) b[k] = std::sqrt((double)k * ((double)k + z));
  }
  gauss_from_jacobi(a, b, s, w);
  for (int k = 0; k < n; ++k) s[k] /= (z + 1.0);
}

static void gauss_tilt_rule_compute(double sigma, int n, std::vector<double>& d, std::vector<double>& w) {
  if (n <= 1 || !(sigma > 0.0)) {
    d.assign(1, 0.0);
    w.assign(1, 1.0);
    return;
  }
  std::vector<double> a(n, 0.0), b(n, 0.0), x, wl;
  for (int k = 1; k < n; ++k) b[k] = (double)k / std::sqrt(4.0 * (double)k * (double)k - 1.0);
  gauss_from_jacobi(a, b, x, wl);
  d.resize(n);
  w.resize(n);
  double sum = 0.0;
  for (int k = 0; k < n; ++k) {
    // symmetrise: Legendre nodes come in +- pairs
    d[k] = 3.0 * sigma * x[k];
    w[k] = wl[k] * std::exp(-(d[k] * d[k]) / (2.0 * sigma * sigma));
    sum += w[k];
  }
  for (int k = 0; k < n; ++k) w[k] /= sum;
}

// Rules are memoised by (kind, parameter bits, n): a dataset-generation loop sets thousands of models that
// share a handful of rules, and the bisection costs ~100 us per 32-node rule.
namespace {
struct RuleKey {
  int kind; uint64_t bits; int n;
  bool operator<(const RuleKey& o) const {
    return kind != o.kind ? kind < o.kind : bits != o.bits ? bits < o.bits : n < o.n;
  }
};
struct Rule { std::vector<double> x, w; };
std::mutex g_rule_mutex;
std::map<RuleKey, Rule> g_rules;

void cached_rule(int kind, double param, int n, std::vector<double>& x, std::vector<double>& w) {
  uint64_t bits;
  std::memcpy(&bits, &param, sizeof bits);
  const RuleKey key{kind, bits, n};
  std::lock_guard<std::mutex> lock(g_rule_mutex);
  auto it = g_rules.find(key);
  if (it == g_rules.end()) {
    Rule r;
    if (kind == 0) schulz_rule_compute(param, n, r.x, r.w); else gauss_tilt_rule_compute(param, n, r.x, r.w);
    if (g_rules.size() >= 4096) g_rules.clear();
    it = g_rules.emplace(key, std::move(r)).first;
  }
  x = it->second.x;
  w = it->second.w;
}
}  // namespace

void schulz_rule(double p, int n, std::vector<double>& s, std::vector<double>& w) { cached_rule(0, p, n, s, w); }
void gauss_tilt_rule(double sigma, int n, std::vector<double>& d, std::vector<double>& w) { cached_rule(1, sigma, n, d, w); }

}  // namespace sas
