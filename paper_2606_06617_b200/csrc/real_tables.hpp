// Host-side (plan-time) tables of the real-space complement and the self term, double precision
// ((S64)-(S68)).
//
// The complement of the mollified kernel is compactly supported: for x = r / r_c < 1
//     L_{p,r_c}(r) = r^-p - S_{p,r_c}(r) = r_c^-p  N_p(x) / x^p,
// with a SMOOTH numerator N_p(x) that follows from SI Props. 2-7 (phi = psi_0^c / psi_0^c(0),
// Phi(x) = int_0^x phi, C0 = Phi(1)):
//     N_1 = 1 - Phi/C0                                   (S17),
//     N_2 = phi                                          (S18)
//     N_3 = 1 - (Phi - x phi)/C0                         (S19),
//     N_4 = phi - x phi'/2                               (S24),
//     N_5 = 1 - (Phi - x phi + x^2 phi'/3)/C0            (S29),
//     N_6 = phi - 5 x phi'/8 + x^2 phi''/8               (S33),
//     N_8, N_10 from Corollary 1 (S57)-(S58), PAPER.md:891-894 (derivatives of phi up to the fourth)
// N_p and dN_p/dx are tabulated as piecewise polynomials (Horner: "the real-space
// kernels G_p" are evaluated the same way as the window); the singular factor x^-p stays explicit.
// Self term: E_self = S_p(0) sum_i q_i^2 / (2 r_c^p) with S_p(0) from (S67); the
// derivatives of phi at 0 come from the moments of psi (S40).
//
// Product code; shares nothing with oracle/.
#pragma once
#include "host_tables.hpp"

namespace pswf {

// psi and its first four derivatives from the Legendre series (three-term recurrence differentiated
// m times: (k+1) P_{k+1}^(m) = (2k+1) (m P_k^(m-1) + x P_k^(m)) - k P_{k-1}^(m))
inline void pswf_eval_d4(const Pswf0& psi, double x, double (&d)[5]) {
  const std::vector<double>& a = psi.leg;
  double p0[5] = {1, 0, 0, 0, 0}, p1[5] = {x, 1, 0, 0, 0};
  for (int m = 0; m < 5; ++m) d[m] = a[0] * p0[m] + (a.size() > 1 ? a[1] * p1[m] : 0.0);
  for (size_t k = 1; k + 1 < a.size(); ++k) {
    double p2[5];
    p2[0] = ((2 * k + 1) * x * p1[0] - k * p0[0]) / (k + 1);
    for (int m = 1; m < 5; ++m) p2[m] = ((2 * k + 1) * (m * p1[m - 1] + x * p1[m]) - k * p0[m]) / (k + 1);
    for (int m = 0; m < 5; ++m) {
      d[m] += a[k + 1] * p2[m];
      p0[m] = p1[m];
      p1[m] = p2[m];
    }
  }
}
inline void pswf_eval_d2(const Pswf0& psi, double x, double& f, double& d1, double& d2) {
  double d[5];
  pswf_eval_d4(psi, x, d);
  f = d[0]; d1 = d[1]; d2 = d[2];
}

struct RealMath {
  const Pswf0& psi;
  GaussLegendre gl;
  explicit RealMath(const Pswf0& p) : psi(p), gl(96) {}
  double Phi(double x) const { return gl.integrate([&](double t) { return psi.eval(t); }, 0.0, x); }
  // numerator N_p(x), 0 <= x <= 1
  double N(int p, double x) const {
    double f, d1, d2;
    pswf_eval_d2(psi, x, f, d1, d2);
    const double C0 = psi.C0;
    switch (p) {
      case 1: return 1.0 - Phi(x) / C0;
      case 2: return f;
      case 3: return 1.0 - (Phi(x) - x * f) / C0;
      case 4: return f - 0.5 * x * d1;
      case 5: return 1.0 - (Phi(x) - x * f + x * x * d1 / 3.0) / C0;
      case 6: return f - 0.625 * x * d1 + 0.125 * x * x * d2;
      case 8: {    // Corollary 1 (S57): N_8 = 1 - x^8 S_8
        double d[5];
        pswf_eval_d4(psi, x, d);
        return d[0] - (11.0 / 16) * x * d[1] + (3.0 / 16) * x * x * d[2] - x * x * x * d[3] / 48;
      }
      case 10: {   // (S58)
        double d[5];
        pswf_eval_d4(psi, x, d);
        const double x2 = x * x;
        return d[0] - (93.0 / 128) * x * d[1] + (29.0 / 128) * x2 * d[2] - (7.0 / 192) * x2 * x * d[3] +
               x2 * x2 * d[4] / 384;
      }
    }
    throw std::invalid_argument("p");
  }
  // psi^(2m)(0) = (-1)^m c^(2m) / lambda_0 * int_{-1}^{1} t^(2m) psi(t) dt     (S40)
  double deriv0(int order) const {
    const int m = order / 2;
    const double mom = 2.0 * gl.integrate([&](double t) { return std::pow(t, order) * psi.eval(t); }, 0.0, 1.0);
    return ((m % 2) ? -1.0 : 1.0) * std::pow(psi.c, order) * mom / psi.lambda0;
  }
  double S0(int p) const {   // (S67)
    const double C0 = psi.C0;
    switch (p) {
      case 1: return 1.0 / C0;
      case 2: return -deriv0(2) / 2.0;
      case 3: return -deriv0(2) / (3.0 * C0);
      case 4: return deriv0(4) / 24.0;
      case 5: return deriv0(4) / (45.0 * C0);
      case 6: return -deriv0(6) / 720.0;
      case 8: return deriv0(8) / 40320.0;        // (S59)
      case 10: return -deriv0(10) / 3628800.0;
    }
    throw std::invalid_argument("p");
  }
};

// Piecewise polynomials for N_p on `panels` uniform panels of x in [0,1]; panel variable
// xi = 2 (x * panels - j) - 1.  coef[(slot * panels + j) * (degree+1) + m] is the xi^m coefficient of
// N_p, dcoef[(slot * panels + j) * degree + m] that of dN_p/dx (the derivative of the SAME polynomial,
// chain factor 2 * panels included).
struct RealTable {
  int panels = 0, degree = 0;
  std::vector<double> coef, dcoef;
  std::vector<double> S0;   // per slot
};

inline RealTable fit_real(const RealMath& rm, const std::vector<int>& distinct_p, int panels, double eps,
                          int max_degree) {
  RealTable tb;
  tb.panels = panels;
  std::vector<std::vector<double>> a;
  int deg = 1;
  for (size_t s = 0; s < distinct_p.size(); ++s) {
    tb.S0.push_back(rm.S0(distinct_p[s]));
    for (int j = 0; j < panels; ++j) {
      a.push_back(ChebFit::coefficients(
          [&](double xi) { return rm.N(distinct_p[s], std::min(1.0, (j + 0.5 * (xi + 1)) / panels)); }));
      deg = std::max(deg, ChebFit::filtered_degree(a.back(), eps, 1.0));   // N_p(0) = 1: scale 1
    }
  }
  deg = std::min(deg, max_degree);
  tb.degree = deg;
  tb.coef.assign(distinct_p.size() * panels * (size_t)(deg + 1), 0.0);
  tb.dcoef.assign(distinct_p.size() * panels * (size_t)deg, 0.0);
  for (size_t s = 0; s < distinct_p.size(); ++s)
    for (int j = 0; j < panels; ++j) {
      std::vector<double> mono = ChebFit::to_monomial(a[s * panels + j], deg);
      for (int m = 0; m <= deg; ++m) tb.coef[(s * panels + j) * (size_t)(deg + 1) + m] = mono[m];
      for (int m = 1; m <= deg; ++m)
        tb.dcoef[(s * panels + j) * (size_t)deg + (m - 1)] = m * mono[m] * 2.0 * panels;
    }
  return tb;
}

}  // namespace pswf
