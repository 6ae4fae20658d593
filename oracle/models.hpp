// oracle/models.hpp -- the four compiled-in models, written out plainly.  TEST INFRASTRUCTURE ONLY.
//
// The paper asks the user for two functions: the member log-likelihood
// log l_i(chi) and the population log-density log f(chi; theta);
// plus a prior on theta (default uniform).  Additive constants independent of chi and
// theta are dropped.  Model table: DESIGN.md section 3.  T is the state precision.
#pragma once
#include <cmath>
#include <cstdint>
#include <limits>
#include <vector>

namespace oracle {

enum Model { M_NORMAL1D = 0, M_THINNED_SCHECHTER1D = 1, M_BINORMAL2D = 2, M_LINREG_ME1D = 3 };

struct Dims { int p, dtheta, n_cols, n_consts; };
inline bool model_dims(int model, Dims* d) {
  switch (model) {
    case M_NORMAL1D:            *d = {1, 2, 2, 0}; return true;   // cols y, sigma;          theta (mu, log tau)
    case M_THINNED_SCHECHTER1D: *d = {1, 3, 2, 6}; return true;   // cols Fhat, g=1/(4 pi r^2); theta (alpha, x*, a)
    case M_BINORMAL2D:          *d = {2, 5, 4, 0}; return true;   // cols y1,y2,s1,s2;       theta (m1,m2,l1,l2,zeta)
    case M_LINREG_ME1D:         *d = {1, 3, 3, 0}; return true;   // cols y, sigma, z;       theta (a, b, log tau)
  }
  return false;
}

// consts of M1: {F_lim, sigma_F, x_lo, x_hi, r_min, r_max}
enum { C_FLIM = 0, C_SIGF = 1, C_XLO = 2, C_XHI = 3, C_RMIN = 4, C_RMAX = 5 };

// ---- member log-likelihood  log l_i(chi) ------------------------------------------------------
template <class T>
inline T loglik(int model, const T* chi, const T* d, const T* consts) {
  switch (model) {
    case M_NORMAL1D:
    case M_LINREG_ME1D: {                       // y ~ N(chi, sigma^2)      (Eq. 3.2 shape)
      const T r = d[0] - chi[0];
      return -(r * r) / (T(2) * d[1] * d[1]);
    }
    case M_THINNED_SCHECHTER1D: {               // Fhat ~ N(L/(4 pi r^2), sigma_F^2), L = e^chi
      const T r = d[0] - d[1] * std::exp(chi[0]);
      return -(r * r) / (T(2) * consts[C_SIGF] * consts[C_SIGF]);
    }
    case M_BINORMAL2D: {                        // independent Gaussian errors per axis
      const T r1 = d[0] - chi[0], r2 = d[1] - chi[1];
      return -T(0.5) * ((r1 * r1) / (d[2] * d[2]) + (r2 * r2) / (d[3] * d[3]));
    }
  }
  return std::numeric_limits<T>::quiet_NaN();
}

// ---- population log-density  log f(chi; theta) ------------------------------------------------
template <class T>
inline T logpop(int model, const T* chi, const T* d, const T* th, const T* consts) {
  switch (model) {
    case M_NORMAL1D: {                          // chi ~ N(mu, tau^2), theta = (mu, lambda = log tau)
      const T r = chi[0] - th[0];
      return -th[1] - T(0.5) * r * r * std::exp(T(-2) * th[1]);
    }
    case M_LINREG_ME1D: {                       // chi ~ N(a + b z, tau^2), theta = (a, b, lambda); middle/right DAG of PAPER.md:117-119
      const T r = chi[0] - th[0] - th[1] * d[2];
      return -th[2] - T(0.5) * r * r * std::exp(T(-2) * th[2]);
    }
    case M_THINNED_SCHECHTER1D: {               // Poisson intensity in x = ln L: A (L/L*)^(alpha+1) e^(-L/L*), truncated
      if (!(chi[0] >= consts[C_XLO] && chi[0] <= consts[C_XHI])) return -std::numeric_limits<T>::infinity();
      const T s = chi[0] - th[1];
      return th[2] + (th[0] + T(1)) * s - std::exp(s);
    }
    case M_BINORMAL2D: {                        // bivariate normal, theta = (m1, m2, l1, l2, zeta), rho = tanh zeta
      const T u1 = (chi[0] - th[0]) * std::exp(-th[2]);
      const T u2 = (chi[1] - th[1]) * std::exp(-th[3]);
      const T ch = std::cosh(th[4]);
      const T rho = std::tanh(th[4]);
      return -th[2] - th[3] + std::log(ch) - ch * ch * (u1 * u1 - T(2) * rho * u1 * u2 + u2 * u2) / T(2);
    }
  }
  return std::numeric_limits<T>::quiet_NaN();
}

// ---- log prior on theta (fp64 always) ---------------------------------------------------------
// Uniform on a wide box ("default uniform"); M1's slope takes the truncated Cauchy of
// PAPER.md:284 (Eq. 5.4) on -2 < alpha < 0.  -inf outside the support.
inline double logprior(int model, const double* th) {
  const double ninf = -std::numeric_limits<double>::infinity();
  switch (model) {
    case M_NORMAL1D:
      if (!(std::fabs(th[0]) <= 1e3 && std::fabs(th[1]) <= 10.0)) return ninf;
      return 0.0;
    case M_LINREG_ME1D:
      if (!(std::fabs(th[0]) <= 1e3 && std::fabs(th[1]) <= 1e3 && std::fabs(th[2]) <= 10.0)) return ninf;
      return 0.0;
    case M_BINORMAL2D:
      if (!(std::fabs(th[0]) <= 1e3 && std::fabs(th[1]) <= 1e3 && std::fabs(th[2]) <= 10.0 &&
            std::fabs(th[3]) <= 10.0 && std::fabs(th[4]) <= 10.0)) return ninf;
      return 0.0;
    case M_THINNED_SCHECHTER1D:
      if (!(th[0] > -2.0 && th[0] < 0.0 && std::fabs(th[1]) <= 20.0 && std::fabs(th[2]) <= 50.0)) return ninf;
      return -std::log(1.0 + th[0] * th[0]);
  }
  return ninf;
}

// ---- Gauss-Legendre rule on [a,b]: nodes are the roots of P_n (Newton), w = 2/((1-x^2) P_n'(x)^2)
inline void gauss_legendre(int n, double a, double b, double* x, double* w) {
  const long double pi = 3.14159265358979323846264338327950288L;
  for (int i = 0; i < n; ++i) {
    long double xi = std::cos(pi * ((long double)i + 0.75L) / ((long double)n + 0.5L));
    long double dp = 0.0L;
    for (int it = 0; it < 100; ++it) {
      long double p0 = 1.0L, p1 = xi;                    // P_0, P_1
      for (int k = 2; k <= n; ++k) {                     // (k) P_k = (2k-1) x P_{k-1} - (k-1) P_{k-2}
        const long double pk = ((2.0L * k - 1.0L) * xi * p1 - (k - 1.0L) * p0) / (long double)k;
        p0 = p1; p1 = pk;
      }
      dp = (long double)n * (xi * p1 - p0) / (xi * xi - 1.0L);   // P_n'
      const long double dx = p1 / dp;
      xi -= dx;
      if (std::fabs((double)dx) < 1e-19) break;
    }
    {   // recompute P_n' at the converged root
      long double p0 = 1.0L, p1 = xi;
      for (int k = 2; k <= n; ++k) {
        const long double pk = ((2.0L * k - 1.0L) * xi * p1 - (k - 1.0L) * p0) / (long double)k;
        p0 = p1; p1 = pk;
      }
      dp = (long double)n * (xi * p1 - p0) / (xi * xi - 1.0L);
    }
    const long double wi = 2.0L / ((1.0L - xi * xi) * dp * dp);
    // roots come out descending in i; store ascending
    const int j = n - 1 - i;
    x[j] = (double)(0.5L * ((long double)b - a) * xi + 0.5L * ((long double)b + a));
    w[j] = (double)(0.5L * ((long double)b - a) * wi);
  }
}

// ---- M1 selection integral (PAPER.md:234 Eq. 4.4 denominator; :363) ---------------------------
// I(alpha, x*) = int dx phi(x) G(x),  G(x) = int_{rmin}^{rmax} dr h(r) eta(F(x,r)),
// h(r) = 3 r^2/(rmax^3 - rmin^3) (uniform in volume), eta(F) = Phi((F - F_lim)/sigma_F)
// (Eq. 5.10 with constant sigma).  sigma_F constant => G does not depend on theta, so the
// 2-D integral collapses to a fixed 1,024-point Gauss-Legendre rule in x with weights W_k = w_k G(x_k);
// G itself by a 256-point rule in r (BASELINE.json configs[1]; reading R9).
struct SelectionTable {
  std::vector<double> xk, Wk;
  void build(const double* c) {
    const int NX = 1024, NR = 256;
    const double four_pi = 12.566370614359172953850573533118;
    xk.assign(NX, 0.0); Wk.assign(NX, 0.0);
    std::vector<double> wx(NX), rk(NR), wr(NR);
    gauss_legendre(NX, c[C_XLO], c[C_XHI], xk.data(), wx.data());
    gauss_legendre(NR, c[C_RMIN], c[C_RMAX], rk.data(), wr.data());
    const double vol = c[C_RMAX] * c[C_RMAX] * c[C_RMAX] - c[C_RMIN] * c[C_RMIN] * c[C_RMIN];
    for (int k = 0; k < NX; ++k) {
      long double G = 0.0L;
      for (int j = 0; j < NR; ++j) {
        const double F = std::exp(xk[k]) / (four_pi * rk[j] * rk[j]);
        const double tt = (F - c[C_FLIM]) / c[C_SIGF];
        const double Phi = 0.5 * std::erfc(-tt / 1.4142135623730950488016887242097);
        G += (long double)(wr[j] * (3.0 * rk[j] * rk[j] / vol) * Phi);
      }
      Wk[k] = wx[k] * (double)G;
    }
  }
  // T(theta) = -e^a sum_k W_k exp((alpha+1)(x_k - x*) - e^(x_k - x*))   (minus the expected detected count)
  double theta_only(const double* th) const {
    long double acc = 0.0L;
    for (size_t k = 0; k < xk.size(); ++k) {
      const double s = xk[k] - th[1];
      acc += (long double)(Wk[k] * std::exp((th[0] + 1.0) * s - std::exp(s)));
    }
    return -std::exp(th[2]) * (double)acc;
  }
};

}  // namespace oracle
