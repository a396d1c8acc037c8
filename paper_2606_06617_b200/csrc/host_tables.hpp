// Host-side (plan-time) mathematics of the PSWF-LR library, double precision.
//
//  * psi_0^c from the prolate ODE in the even Legendre basis ((S37)-(S41));
//  * the Fourier-side kernels of SI Theorem 1 (S47)-(S52), split as
//    "bare transform x / + smooth part" so that only smooth functions T_p(x),
//    x = k r_c / c in [0,1], are tabulated;
//  * piecewise-polynomial (Horner) tables for the window and for T_p with the degree chosen by
//    Chebyshev-coefficient filtering: expand on a degree-40 Chebyshev basis,
//    drop |a_n| <= 0.01 eps max|a_m|, convert to monomials.
//
// Product code.  Independent of oracle/ (which is numpy); nothing here is shared with it.
#pragma once
#include <algorithm>
#include <cmath>
#include <stdexcept>
#include <vector>

namespace pswf {

constexpr double kPi = 3.14159265358979323846;

// ---- Gauss-Legendre nodes on [-1,1] ---------------------------------------------------------
struct GaussLegendre {
  std::vector<double> x, w;
  explicit GaussLegendre(int n) : x(n), w(n) {
    for (int i = 0; i < n; ++i) {
      double t = std::cos(kPi * (i + 0.75) / (n + 0.5));
      double dp = 0;
      for (int it = 0; it < 100; ++it) {
        double p0 = 1, p1 = t;
        for (int k = 1; k < n; ++k) {
          double p2 = ((2 * k + 1) * t * p1 - k * p0) / (k + 1);
          p0 = p1; p1 = p2;
        }
        dp = n * (t * p1 - p0) / (t * t - 1);
        double dt = p1 / dp;
        t -= dt;
        if (std::fabs(dt) < 1e-16) break;
      }
      x[i] = t;
      w[i] = 2 / ((1 - t * t) * dp * dp);
    }
  }
  template <class F> double integrate(F f, double a, double b) const {
    double s = 0, hm = 0.5 * (b - a), mid = 0.5 * (b + a);
    for (size_t i = 0; i < x.size(); ++i) s += w[i] * f(mid + hm * x[i]);
    return s * hm;
  }
};

// ---- order-zero PSWF ------------------------------------------------------------------------
struct Pswf0 {
  double c = 0, lambda0 = 0, C0 = 0;
  std::vector<double> leg;  // psi(x) = sum_k leg[k] P_k(x), odd entries zero, psi(0) = 1

  explicit Pswf0(double c_) : c(c_) {
    const int n = (int)(2 * c) + 48;  // even terms k = 0,2,..,2(n-1)
    std::vector<double> d(n), e(n, 0.0);
    for (int i = 0; i < n; ++i) {
      double k = 2.0 * i;
      d[i] = k * (k + 1) + c * c * (2 * k * (k + 1) - 1) / ((2 * k + 3) * (2 * k - 1));
      if (i + 1 < n)
        e[i] = c * c * (k + 1) * (k + 2) / ((2 * k + 3) * std::sqrt((2 * k + 1) * (2 * k + 5)));
    }
    // A is symmetric positive definite (it is the matrix of -d/dx(1-x^2)d/dx + c^2 x^2); its
    // lowest eigenvector is psi_0.  Inverse iteration (Thomas solves), then Rayleigh polishing.
    std::vector<double> v(n, 0.0), y(n), cp(n), dpv(n);
    for (int i = 0; i < n; ++i) v[i] = std::exp(-0.5 * i);
    auto solve = [&](double shift) {
      cp[0] = e[0] / (d[0] - shift);
      dpv[0] = v[0] / (d[0] - shift);
      for (int i = 1; i < n; ++i) {
        double m = (d[i] - shift) - e[i - 1] * cp[i - 1];
        cp[i] = e[i] / m;
        dpv[i] = (v[i] - e[i - 1] * dpv[i - 1]) / m;
      }
      y[n - 1] = dpv[n - 1];
      for (int i = n - 2; i >= 0; --i) y[i] = dpv[i] - cp[i] * y[i + 1];
      double nrm = 0;
      for (double t : y) nrm += t * t;
      nrm = std::sqrt(nrm);
      for (int i = 0; i < n; ++i) v[i] = y[i] / nrm;
    };
    for (int it = 0; it < 80; ++it) solve(0.0);
    // coefficients in the un-normalised P_k basis
    leg.assign(2 * n - 1, 0.0);
    for (int i = 0; i < n; ++i) leg[2 * i] = v[i] * std::sqrt(2.0 * i + 0.5);
    double v0 = eval(0.0);
    for (double& t : leg) t /= v0;
    C0 = leg[0];            // int_0^1 psi = (1/2) int_{-1}^{1} psi = leg[0]
    lambda0 = 2 * leg[0];   // (S41)
  }

  double eval(double x) const {
    double p0 = 1, p1 = x, s = leg[0] + (leg.size() > 1 ? leg[1] * x : 0.0);
    for (size_t k = 1; k + 1 < leg.size(); ++k) {
      double p2 = ((2 * k + 1) * x * p1 - k * p0) / (k + 1);
      s += leg[k + 1] * p2;
      p0 = p1; p1 = p2;
    }
    return s;
  }
};

// ---- Chebyshev fit of f on [-1,1], filtered, in monomials -------------------------------------
struct ChebFit {
  static constexpr int kBasis = 40;  // PAPER.md:329 "fixed high-order Chebyshev basis (up to degree 40)"
  // Chebyshev coefficients a_0..a_40 of f sampled at the 41 Chebyshev-Gauss nodes.
  template <class F> static std::vector<double> coefficients(F f) {
    const int N = kBasis + 1;
    std::vector<double> fx(N), a(N);
    for (int j = 0; j < N; ++j) fx[j] = f(std::cos(kPi * (j + 0.5) / N));
    for (int n = 0; n < N; ++n) {
      double s = 0;
      for (int j = 0; j < N; ++j) s += fx[j] * std::cos(kPi * n * (j + 0.5) / N);
      a[n] = s * 2.0 / N;
    }
    a[0] *= 0.5;
    return a;
  }
  // highest degree kept by the filter |a_n| <= 0.01 eps max|a_m|, relative to `scale`
  static int filtered_degree(const std::vector<double>& a, double eps, double scale) {
    int deg = 0;
    for (int n = 0; n < (int)a.size(); ++n)
      if (std::fabs(a[n]) > 0.01 * eps * scale) deg = n;
    return deg;
  }
  // monomial coefficients (in xi) of sum_{n<=deg} a_n T_n(xi)
  static std::vector<double> to_monomial(const std::vector<double>& a, int deg) {
    std::vector<double> out(deg + 1, 0.0), t0(deg + 1, 0.0), t1(deg + 1, 0.0), t2(deg + 1, 0.0);
    t0[0] = 1;
    out[0] += a[0];
    if (deg >= 1) { t1[1] = 1; out[1] += a[1]; }
    for (int n = 2; n <= deg; ++n) {
      std::fill(t2.begin(), t2.end(), 0.0);
      for (int k = 0; k < deg; ++k) t2[k + 1] += 2 * t1[k];
      for (int k = 0; k <= deg; ++k) t2[k] -= t0[k];
      for (int k = 0; k <= deg; ++k) out[k] += a[n] * t2[k];
      t0 = t1; t1 = t2;
    }
    return out;
  }
};

// ---- window tables -----------------------------------------------------------------------------
// Panel t (t = 0..w-1) covers window arguments z = 2 (t + delta)/w - 1, delta in [0,1) (DESIGN.md
// reading R4); the panel variable is xi = 2 delta - 1.  coef[m * w + t] is the xi^m coefficient.
struct WindowTable {
  int w = 0, degree = 0;
  std::vector<double> coef;   // (degree+1) x w
  std::vector<double> dcoef;  // derivative w.r.t. xi, degree x w  (d/dxi of the SAME polynomial)
};

inline WindowTable fit_window(const Pswf0& psi, int w, double eps, int max_degree) {
  WindowTable tb;
  tb.w = w;
  std::vector<std::vector<double>> a(w);
  int deg = 1;
  for (int t = 0; t < w; ++t) {
    a[t] = ChebFit::coefficients([&](double xi) { return psi.eval(2.0 * (t + 0.5 * (xi + 1)) / w - 1.0); });
    deg = std::max(deg, ChebFit::filtered_degree(a[t], eps, 1.0));  // scale: psi(0) = 1
  }
  deg = std::min(deg, max_degree);
  tb.degree = deg;
  tb.coef.assign((size_t)(deg + 1) * w, 0.0);
  tb.dcoef.assign((size_t)deg * w, 0.0);
  for (int t = 0; t < w; ++t) {
    std::vector<double> mono = ChebFit::to_monomial(a[t], deg);
    for (int m = 0; m <= deg; ++m) tb.coef[(size_t)m * w + t] = mono[m];
    for (int m = 1; m <= deg; ++m) tb.dcoef[(size_t)(m - 1) * w + t] = m * mono[m];
  }
  return tb;
}

// ---- Fourier-side kernels ------------------------------------------------------------------------
// S^_p(kappa) = pre_p(kappa) * T_p(x) + log_p(x),  x = kappa / c  (Theorem 1, (S47)-(S52)):
//   p=1: (4 pi / kappa^2) T_1,                 T_1 = phi(x)
//   p=2: (2 pi^2 / kappa) T_2,                 T_2 = 1 - A(x),            A = (1/C0) int_0^x phi
//   p=3: 4 pi (T_3 - ln x),                    T_3 = int_x^1 (phi - 1)/t dt
//   p=4: pi^2 c T_4,                           T_4 = J_1/C0 - x (1 - A),  J_n = int_x^1 t^n phi
//   p=5: (2 pi c^2 / 3)(T_5 + x^2 ln x),       T_5 = J_1 - x^2 T_3
//   p=6: (pi^2 c^3 / 12) T_6,                  T_6 = x^3 (1 - A) - 3 x^2 J_1 / (2 C0) + J_3 / (2 C0)
//   p=8: (pi^2 c^5 / 72) T_8,   p=10: (pi^2 c^7 / 576) T_10   (SI Section 6, see T())
// and Phi^_p(k) = r_c^(3-p) S^_p(k r_c)  (S60).
struct KernelMath {
  const Pswf0& psi;
  GaussLegendre gl;
  explicit KernelMath(const Pswf0& p) : psi(p), gl(96) {}
  double A(double x) const { return gl.integrate([&](double t) { return psi.eval(t); }, 0.0, x) / psi.C0; }
  double J(int n, double x) const {
    return gl.integrate([&](double t) { return std::pow(t, n) * psi.eval(t); }, x, 1.0);
  }
  double Llog(double x) const {
    return gl.integrate([&](double t) { return (psi.eval(t) - 1.0) / t; }, x, 1.0);
  }
  double T(int p, double x) const {
    switch (p) {
      case 1: return psi.eval(x);
      case 2: return 1.0 - A(x);
      case 3: return Llog(x);
      case 4: return J(1, x) / psi.C0 - x * (1.0 - A(x));
      case 5: return J(1, x) - x * x * Llog(x);
      case 6: return x * x * x * (1.0 - A(x)) - 1.5 * x * x * J(1, x) / psi.C0 + 0.5 * J(3, x) / psi.C0;
      // p = 8, 10: (S56) applied to (S52) and once more, integrals over [k, c] by the
      // truncation convention; with int_x^1 y^m J_n = (J_{m+n+1} - x^{m+1} J_n) / (m+1) and 1 - A = J_0 / C0:
      //   S^_8  = (pi^2 c^5 / 72)  T_8,   S^_10 = (pi^2 c^7 / 576) T_10
      case 8: {
        const double x2 = x * x, x4 = x2 * x2;
        return (-x4 * x * J(0, x) / 5 + 0.375 * x4 * J(1, x) - 0.25 * x2 * J(3, x) + 0.075 * J(5, x)) / psi.C0;
      }
      case 10: {
        const double x2 = x * x, x4 = x2 * x2, x6 = x4 * x2;
        return (x6 * x * J(0, x) / 35 - x6 * J(1, x) / 16 + x4 * J(3, x) / 16 - 0.0375 * x2 * J(5, x) +
                J(7, x) / 112) / psi.C0;
      }
    }
    throw std::invalid_argument("p");
  }
  // zero-mode constants Phi0_p with E_0 = Phi0 Q_net^2 / (2V)
  double Phi0(int p, double r_c) const {
    const double c = psi.c, C0 = psi.C0;
    switch (p) {
      case 1:  // (S72)-(S73), E_IB = 0
        return -(2 * kPi * r_c * r_c / C0) * gl.integrate([&](double u) { return u * u * psi.eval(u); }, 0.0, 1.0);
      case 2: return -4 * kPi * r_c * C0;                               // (S74)-(S75)
      case 3: return 4 * kPi * (std::log(c / r_c) + Llog(0.0));         // (S77)-(S78)
      case 4: return std::pow(r_c, -1.0) * kPi * kPi * c * T(4, 0.0);   // (S79): k -> 0 of (S50)
      case 5: return std::pow(r_c, -2.0) * (2 * kPi * c * c / 3) * T(5, 0.0);
      case 6: return std::pow(r_c, -3.0) * (kPi * kPi * c * c * c / 12) * T(6, 0.0);
      case 8: return std::pow(r_c, -5.0) * (kPi * kPi * std::pow(c, 5) / 72) * T(8, 0.0);
      case 10: return std::pow(r_c, -7.0) * (kPi * kPi * std::pow(c, 7) / 576) * T(10, 0.0);
    }
    throw std::invalid_argument("p");
  }
};

// Piecewise polynomials for T_p on `panels` uniform panels of x in [0,1]; panel variable
// xi = 2 (x * panels - j) - 1.  coef[(p_slot * panels + j) * (degree+1) + m].
struct KernelTable {
  int panels = 0, degree = 0;
  std::vector<int> exponents;   // distinct p, ascending
  std::vector<double> coef;
};

inline KernelTable fit_kernels(const KernelMath& km, const std::vector<int>& distinct_p, int panels,
                               double eps, int max_degree) {
  KernelTable tb;
  tb.panels = panels;
  tb.exponents = distinct_p;
  std::vector<std::vector<double>> a;
  std::vector<double> scale(distinct_p.size(), 0.0);
  int deg = 1;
  for (size_t s = 0; s < distinct_p.size(); ++s)
    for (int j = 0; j < panels; ++j) {
      a.push_back(ChebFit::coefficients(
          [&](double xi) { return km.T(distinct_p[s], (j + 0.5 * (xi + 1)) / panels); }));
      for (double v : a.back()) scale[s] = std::max(scale[s], std::fabs(v));
    }
  for (size_t s = 0; s < distinct_p.size(); ++s)
    for (int j = 0; j < panels; ++j)
      deg = std::max(deg, ChebFit::filtered_degree(a[s * panels + j], eps, scale[s]));
  deg = std::min(deg, max_degree);
  tb.degree = deg;
  tb.coef.assign(distinct_p.size() * panels * (size_t)(deg + 1), 0.0);
  for (size_t s = 0; s < distinct_p.size(); ++s)
    for (int j = 0; j < panels; ++j) {
      std::vector<double> mono = ChebFit::to_monomial(a[s * panels + j], deg);
      for (int m = 0; m <= deg; ++m) tb.coef[(s * panels + j) * (size_t)(deg + 1) + m] = mono[m];
    }
  return tb;
}

}  // namespace pswf
