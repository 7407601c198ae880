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
static void legendre_rule_01_compute(int n, std::vector<double>& x, std::vector<double>& w);
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
    if (kind == 0) schulz_rule_compute(param, n, r.x, r.w);
    else if (kind == 1) gauss_tilt_rule_compute(param, n, r.x, r.w);
    else legendre_rule_01_compute(n, r.x, r.w);
    if (g_rules.size() >= 4096) g_rules.clear();
    it = g_rules.emplace(key, std::move(r)).first;
  }
  x = it->second.x;
  w = it->second.w;
}
}  // namespace

void schulz_rule(double p, int n, std::vector<double>& s, std::vector<double>& w) { cached_rule(0, p, n, s, w); }
void gauss_tilt_rule(double sigma, int n, std::vector<double>& d, std::vector<double>& w) { cached_rule(1, sigma, n, d, w); }

static void legendre_rule_01_compute(int n, std::vector<double>& x, std::vector<double>& w) {
  std::vector<double> a(n, 0.0), b(n, 0.0), xs, ws;
  for (int k = 1; k < n; ++k) b[k] = (double)k / std::sqrt(4.0 * (double)k * (double)k - 1.0);
  gauss_from_jacobi(a, b, xs, ws);   // on [-1, 1], weights summing to 1
  x.resize(n);
  w.resize(n);
  for (int i = 0; i < n; ++i) { x[i] = 0.5 * (xs[i] + 1.0); w[i] = ws[i]; }
}

void legendre_rule_01(int n, std::vector<double>& x, std::vector<double>& w) { cached_rule(2, 0.0, n, x, w); }

namespace {

struct MsaRule {
  std::vector<double> x, w;   // 64 nodes on [0, 1]
};

inline double msa_qin(double x, double a, double b, double E, double Cp, double k) {
  return ((0.5 * a) * (x * x - 1.0) + b * (x - 1.0)) + (E * std::exp(-k * x) - Cp);
}

// the five equations for u = (a, b, E, C', H'): coefficients of x, 1 and exp(-kx) of Baxter's relation for x h(x)
// inside the core (h = -1), the closure c = -beta u outside, and the Laplace transform at k of the same relation
// outside the core, which ties H' = int_1^inf t h(t) exp(-k (t - 1)) dt to the rest (DESIGN.md R-S2)
void msa_residual(const double u[5], double eta, double gam, double k, const MsaRule& R, double r[5]) {
  const double a = u[0], b = u[1], E = u[2], Cp = u[3], Hp = u[4];
  const double e = std::exp(-k), Dp = E * e - Cp;
  const int n = (int)R.x.size();
  double I0 = 0.0, I1 = 0.0, Qt = 0.0;
  for (int i = 0; i < n; ++i) {
    const double q = msa_qin(R.x[i], a, b, E, Cp, k);
    I0 += R.w[i] * q;
    I1 += R.w[i] * R.x[i] * q;
    Qt += R.w[i] * q * std::exp(-k * R.x[i]);
  }
  r[0] = a - (1.0 - 12.0 * eta * (I0 + Dp / k));
  r[1] = b - 12.0 * eta * (I1 + Dp * (1.0 / k + 1.0 / (k * k)));
  r[2] = -k * E + 12.0 * eta * Dp * ((1.0 + k) / (k * k) + Hp);
  r[3] = k * Dp * (1.0 - 12.0 * eta * (Qt + Dp * e / (2.0 * k))) + gam;
  const double phi1 = (1.0 - e * (1.0 + k)) / (k * k);
  double T = Dp * phi1 / (2.0 * k);
  for (int i = 0; i < n; ++i) {
    const double y = R.x[i];
    double G = Dp * e / (2.0 * k);
    for (int j = 0; j < n; ++j) {
      const double s = y + (1.0 - y) * R.x[j];
      G += (1.0 - y) * R.w[j] * msa_qin(s, a, b, E, Cp, k) * std::exp(-k * s);
    }
    T += R.w[i] * (-(1.0 - y)) * std::exp(k * y) * G;
  }
  r[4] = Hp * (1.0 - 12.0 * eta * Qt) - Dp / 2.0 - 12.0 * eta * T;
}

// 5 x 5 linear system by Gaussian elimination with partial pivoting; false if singular
bool solve5(double A[5][5], double rhs[5], double x[5]) {
  int p[5] = {0, 1, 2, 3, 4};
  for (int c = 0; c < 5; ++c) {
    int best = c;
    for (int r = c + 1; r < 5; ++r)
      if (std::fabs(A[p[r]][c]) > std::fabs(A[p[best]][c])) best = r;
    std::swap(p[c], p[best]);
    const double piv = A[p[c]][c];
    if (!(std::fabs(piv) > 0.0)) return false;
    for (int r = c + 1; r < 5; ++r) {
      const double f = A[p[r]][c] / piv;
      for (int cc = c; cc < 5; ++cc) A[p[r]][cc] -= f * A[p[c]][cc];
      rhs[p[r]] -= f * rhs[p[c]];
    }
  }
  for (int c = 4; c >= 0; --c) {
    double s = rhs[p[c]];
    for (int cc = c + 1; cc < 5; ++cc) s -= A[p[c]][cc] * x[cc];
    x[c] = s / A[p[c]][c];
  }
  return true;
}

}  // namespace

static bool msa_solve_compute(double eta, double gam, double k, double out[5], double* g_contact) {
  MsaRule R;
  legendre_rule_01(64, R.x, R.w);
  double u[5] = {(1.0 + 2.0 * eta) / ((1.0 - eta) * (1.0 - eta)), -1.5 * eta / ((1.0 - eta) * (1.0 - eta)), 0.0, 0.0, 0.0};
  const int steps = 20;
  for (int s = 0; s <= steps; ++s) {
    const double g = gam * (double)s / (double)steps;
    for (int it = 0; it < 60; ++it) {
      double r[5], J[5][5];
      msa_residual(u, eta, g, k, R, r);
      for (int j = 0; j < 5; ++j) {   // central differences: the equations are at most quadratic in u
        const double h = 1.0e-6 * std::max(1.0, std::fabs(u[j]));
        double up[5], um[5], rp[5], rm[5];
        for (int i = 0; i < 5; ++i) { up[i] = u[i]; um[i] = u[i]; }
        up[j] += h; um[j] -= h;
        msa_residual(up, eta, g, k, R, rp);
        msa_residual(um, eta, g, k, R, rm);
        for (int i = 0; i < 5; ++i) J[i][j] = (rp[i] - rm[i]) / (2.0 * h);
      }
      double rhs[5], st[5];
      for (int i = 0; i < 5; ++i) rhs[i] = -r[i];
      if (!solve5(J, rhs, st)) return false;
      double smax = 0.0, umax = 1.0;
      for (int i = 0; i < 5; ++i) { u[i] += st[i]; smax = std::max(smax, std::fabs(st[i])); umax = std::max(umax, std::fabs(u[i])); }
      if (!std::isfinite(smax)) return false;
      if (smax < 1.0e-15 * umax) break;
    }
  }
  double r[5], rmax = 0.0;
  msa_residual(u, eta, gam, k, R, r);
  for (int i = 0; i < 5; ++i) rmax = std::max(rmax, std::fabs(r[i]));
  if (!(rmax < 1.0e-11)) return false;
  out[0] = u[0]; out[1] = u[1]; out[2] = u[2]; out[3] = u[3]; out[4] = u[2] * std::exp(-k) - u[3];
  if (g_contact) *g_contact = u[0] + u[1] - k * u[3];
  return true;
}

// The closure costs ~45 ms to solve (20 continuation steps of Newton's method, each residual a 64 x 64 double
// sum); a fitting or dataset loop sets the same charged system again and again: memoised by the three parameters.
namespace {
struct MsaKey {
  uint64_t a, b, c;
  bool operator<(const MsaKey& o) const { return a != o.a ? a < o.a : b != o.b ? b < o.b : c < o.c; }
};
struct MsaSol { bool ok; double u[5]; double g1; };
std::mutex g_msa_mutex;
std::map<MsaKey, MsaSol> g_msa;
}  // namespace

bool msa_solve(double eta, double gam, double k, double out[5], double* g_contact) {
  MsaKey key;
  std::memcpy(&key.a, &eta, 8);
  std::memcpy(&key.b, &gam, 8);
  std::memcpy(&key.c, &k, 8);
  std::lock_guard<std::mutex> lock(g_msa_mutex);
  auto it = g_msa.find(key);
  if (it == g_msa.end()) {
    MsaSol sol{};
    sol.ok = msa_solve_compute(eta, gam, k, sol.u, &sol.g1);
    if (g_msa.size() >= 1024) g_msa.clear();
    it = g_msa.emplace(key, sol).first;
  }
  for (int i = 0; i < 5; ++i) out[i] = it->second.u[i];
  if (g_contact) *g_contact = it->second.g1;
  return it->second.ok;
}

}  // namespace sas
