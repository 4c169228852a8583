// cosmology.cpp -- background functions of the FastPM operators, host float64.
// The paper prints only Eq. 1-2 and defers the modified kick/drift operators to
// Feng et al. 2016; the growth-factor form used here is derived in DESIGN.md
// (reading R4): demand that a Zel'dovich flow x = q + D1(a) psi is reproduced exactly.
//   G = a^3 E dD/da;  dD1/da = G1/(a^3 E), dG1/da = 1.5 Om D1/(a^2 E),
//                     dD2/da = G2/(a^3 E), dG2/da = 1.5 Om (D2 - D1^2)/(a^2 E)
//   Drift(ai, ac, af) = [D1(af) - D1(ai)] / Gf(ac),   Gf = a^3 E dD1/da (D1 normalised to D1(1)=1)
//   Kick (ai, ac, af) = [Gf(af) - Gf(ai)] / (1.5 Om D1(ac))
#include <cmath>
#include <map>
#include <mutex>
#include <utility>

#include "fpm_internal.h"

namespace fpm {

namespace {

struct State { double d1, g1, d2, g2; };

inline double hubble(double om, double a) { return std::sqrt(om / (a * a * a) + (1.0 - om)); }

// derivatives with respect to s = ln a
inline State deriv(double om, double s, const State& y) {
  const double a = std::exp(s), e = hubble(om, a);
  const double ia2e = 1.0 / (a * a * e);       // a d/da of D: G / (a^2 E)
  const double src = 1.5 * om / (a * e);       // a * 1.5 Om / (a^2 E)
  return State{y.g1 * ia2e, src * y.d1, y.g2 * ia2e, src * (y.d2 - y.d1 * y.d1)};
}

inline State axpy(const State& y, double h, const State& k) {
  return State{y.d1 + h * k.d1, y.g1 + h * k.g1, y.d2 + h * k.d2, y.g2 + h * k.g2};
}

// Integrate from deep matter domination (D1 = a, D2 = -3/7 a^2) to a_end, RK4 in ln a.
State integrate(double om, double a_end) {
  const double a0 = 1e-5;
  const double e0 = hubble(om, a0);
  State y{a0, a0 * a0 * a0 * e0, -3.0 / 7.0 * a0 * a0, a0 * a0 * a0 * e0 * (-6.0 / 7.0 * a0)};
  const double s0 = std::log(a0), s1 = std::log(a_end);
  const int steps = 1 << 14;
  const double h = (s1 - s0) / steps;
  double s = s0;
  for (int i = 0; i < steps; ++i) {
    const State k1 = deriv(om, s, y);
    const State k2 = deriv(om, s + 0.5 * h, axpy(y, 0.5 * h, k1));
    const State k3 = deriv(om, s + 0.5 * h, axpy(y, 0.5 * h, k2));
    const State k4 = deriv(om, s + h, axpy(y, h, k3));
    y.d1 += h / 6.0 * (k1.d1 + 2.0 * (k2.d1 + k3.d1) + k4.d1);
    y.g1 += h / 6.0 * (k1.g1 + 2.0 * (k2.g1 + k3.g1) + k4.g1);
    y.d2 += h / 6.0 * (k1.d2 + 2.0 * (k2.d2 + k3.d2) + k4.d2);
    y.g2 += h / 6.0 * (k1.g2 + 2.0 * (k2.g2 + k3.g2) + k4.g2);
    s += h;
  }
  return y;
}

std::mutex g_mu;
std::map<std::pair<double, double>, State> g_cache;

State integrate_cached(double om, double a) {
  std::lock_guard<std::mutex> lock(g_mu);
  auto key = std::make_pair(om, a);
  auto it = g_cache.find(key);
  if (it != g_cache.end()) return it->second;
  const State y = integrate(om, a);
  if (g_cache.size() > 4096) g_cache.clear();
  g_cache[key] = y;
  return y;
}

// int_ai^af da / (a^pw E) with Gauss-Legendre (8 points on 64 panels)
double quinn(double om, double ai, double af, int pw) {
  static const double xs[4] = {0.1834346424956498, 0.5255324099163290, 0.7966664774136267,
                               0.9602898564975363};
  static const double ws[4] = {0.3626837833783620, 0.3137066458778873, 0.2223810344533745,
                               0.1012285362903763};
  const int panels = 64;
  const double w = (af - ai) / panels;
  double sum = 0.0;
  for (int i = 0; i < panels; ++i) {
    const double mid = ai + (i + 0.5) * w;
    for (int j = 0; j < 4; ++j)
      for (int sgn = -1; sgn <= 1; sgn += 2) {
        const double a = mid + sgn * 0.5 * w * xs[j];
        sum += ws[j] * 0.5 * w / (std::pow(a, pw) * hubble(om, a));
      }
  }
  return sum;
}

}  // namespace

GrowthOut growth(double om, double a) {
  const State y = integrate_cached(om, a), y1 = integrate_cached(om, 1.0);
  GrowthOut g;
  g.E = hubble(om, a);
  g.D1 = y.d1 / y1.d1;
  g.D2 = y.d2 / (y1.d1 * y1.d1);
  g.Gf = y.g1 / y1.d1;
  g.f1 = y.g1 / (a * a * g.E * y.d1);
  g.f2 = y.g2 / (a * a * g.E * y.d2);
  g.gf = 1.5 * om * g.D1 / (a * a * g.E);
  return g;
}

double drift_factor(double om, double ai, double ac, double af, int factor_mode) {
  if (factor_mode == FPM_FACTORS_QUINN) return quinn(om, ai, af, 3);
  return (growth(om, af).D1 - growth(om, ai).D1) / growth(om, ac).Gf;
}

double kick_factor(double om, double ai, double ac, double af, int factor_mode) {
  if (factor_mode == FPM_FACTORS_QUINN) return quinn(om, ai, af, 2);
  return (growth(om, af).Gf - growth(om, ai).Gf) / (1.5 * om * growth(om, ac).D1);
}

}  // namespace fpm
