// oracle/models.hpp -- the six compiled-in models, written out plainly.  TEST INFRASTRUCTURE ONLY.
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

enum Model { M_NORMAL1D = 0, M_THINNED_SCHECHTER1D = 1, M_BINORMAL2D = 2, M_LINREG_ME1D = 3, M_BB1_FLUXNOISE1D = 4,
             M_NORMAL3D_KNOWNCOV = 5,
             // the same normal-normal model for p-vector latents, p = 4, 5, 6 (RAM of Eq. 2.6 is stated for any dimension,
             // PAPER.md:129-140; section 3 is its p = 3 instance): chi ~ N_p(mu, C_pop), y_j ~ N(chi_j, sigma_j^2)
             M_NORMAL4D_KNOWNCOV = 6, M_NORMAL5D_KNOWNCOV = 7, M_NORMAL6D_KNOWNCOV = 8 };

// latent dimension of the normal-normal family (0 for the other models)
inline int normal_family_p(int model) {
  return (model >= M_NORMAL3D_KNOWNCOV && model <= M_NORMAL6D_KNOWNCOV) ? model - M_NORMAL3D_KNOWNCOV + 3 : 0;
}

struct Dims { int p, dtheta, n_cols, n_consts; };
inline bool model_dims(int model, Dims* d) {
  switch (model) {
    case M_NORMAL1D:            *d = {1, 2, 2, 0}; return true;   // cols y, sigma;          theta (mu, log tau)
    case M_THINNED_SCHECHTER1D: *d = {1, 3, 2, 6}; return true;   // cols Fhat, g=1/(4 pi r^2); theta (alpha, x*, a)
    case M_BINORMAL2D:          *d = {2, 5, 4, 0}; return true;   // cols y1,y2,s1,s2;       theta (m1,m2,l1,l2,zeta)
    case M_LINREG_ME1D:         *d = {1, 3, 3, 0}; return true;   // cols y, sigma, z;       theta (a, b, log tau)
    case M_BB1_FLUXNOISE1D:     *d = {1, 3, 2, 7}; return true;   // cols Fhat, g=1/(4 pi r^2); theta (beta, ln l, ln u)
    case M_NORMAL3D_KNOWNCOV:   *d = {3, 3, 3, 9}; return true;   // cols y1, y2, y3;        theta = mu (3)
    case M_NORMAL4D_KNOWNCOV:   *d = {4, 4, 4, 14}; return true;  // cols y1..y4;  theta = mu;  consts sigma_1..4, C_pop (10)
    case M_NORMAL5D_KNOWNCOV:   *d = {5, 5, 5, 20}; return true;
    case M_NORMAL6D_KNOWNCOV:   *d = {6, 6, 6, 27}; return true;
  }
  return false;
}

// consts of M1: {F_lim, sigma_F, x_lo, x_hi, r_min, r_max}
enum { C_FLIM = 0, C_SIGF = 1, C_XLO = 2, C_XHI = 3, C_RMIN = 4, C_RMAX = 5 };
// consts of M4 (the paper's case study): {sigma_0, alpha (the noise slope of Eq. 5.8), x_lo, x_hi,
// r_min, r_max, F_th}; x_lo .. r_max sit at the same indices as in M1
enum { B_SIG0 = 0, B_ANOISE = 1, B_FTH = 6 };

// consts of the normal-normal family (the benchmark of PAPER.md:146-166, Eq. 3.1-3.4, for p = 3 .. 6): {sigma_1 .. sigma_p,
// then the packed lower triangle of C_pop row-major: C11, C21, C22, C31, ...}; C_pop and sigma_j are KNOWN, theta = mu
// (PAPER.md:166).  The covariance block starts at index p.
enum { N3_SIG = 0 };

// log C(beta, u, l), the BB1 normaliser of PAPER.md:429 (Eq. C.3):
//   C = 1 / (Gamma(beta+1) (1 - (1 + u/l)^-(beta+1)))   (beta > -2, beta != -1),     C = 1/log(1 + u/l)  (beta = -1).
// For -2 < beta < -1 both factors are negative, the product is positive; near beta = -1 each factor keeps its
// relative accuracy (lgamma; expm1/log1p), so the 0 x inf product is harmless.
inline double bb1_log_norm(double beta, double l, double u) {
  const double b1 = beta + 1.0;
  const double A = std::log1p(u / l);
  if (b1 == 0.0) return -std::log(A);
  const double q = -std::expm1(-b1 * A);              // 1 - (1 + u/l)^-(beta+1)
  return -(std::lgamma(b1) + std::log(std::fabs(q)));
}

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
    case M_NORMAL3D_KNOWNCOV: case M_NORMAL4D_KNOWNCOV: case M_NORMAL5D_KNOWNCOV: case M_NORMAL6D_KNOWNCOV: {
      // y_ij ~ N(chi_ij, sigma_j^2), j = 1..p   (Eq. 3.2, sigma_j of :164)
      const int np = normal_family_p(model);
      T s = T(0);
      for (int j = 0; j < np; ++j) { const T r = d[j] - chi[j]; s += (r * r) / (consts[N3_SIG + j] * consts[N3_SIG + j]); }
      return -T(0.5) * s;
    }
    case M_BB1_FLUXNOISE1D: {
      // Fhat ~ N(F, sigma(F)^2), sigma(F)^2 = sigma_0^2 + (alpha F)^2 (Eq. 5.8), F = L/(4 pi r^2),
      // L = e^chi; the member likelihood is the sampling density as a function of F -- the g(n_obs; F) choice
      // of PAPER.md:298-321 (Eq. 5.6), NOT Gaussian in F: the 1/sigma(F) factor stays.
      const T F = d[1] * std::exp(chi[0]);
      const T s2 = consts[B_SIG0] * consts[B_SIG0] + (consts[B_ANOISE] * F) * (consts[B_ANOISE] * F);
      const T r = d[0] - F;
      return -T(0.5) * std::log(s2) - (r * r) / (T(2) * s2);
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
    case M_NORMAL3D_KNOWNCOV: case M_NORMAL4D_KNOWNCOV: case M_NORMAL5D_KNOWNCOV: case M_NORMAL6D_KNOWNCOV: {
      // chi ~ N(mu, C_pop) (Eq. 3.1), C_pop known: log f = -1/2 (chi - mu)^T C_pop^-1 (chi - mu) + const.
      // Plain route: factor C_pop = G G^T (Cholesky), solve G w = chi - mu, then -1/2 w^T w.
      const int np = normal_family_p(model);
      T G[6][6] = {};
      const T* Cp = consts + np;
      for (int r = 0; r < np; ++r)
        for (int k = 0; k <= r; ++k) {
          T a = Cp[r * (r + 1) / 2 + k];
          for (int m = 0; m < k; ++m) a -= G[r][m] * G[k][m];
          G[r][k] = (r == k) ? std::sqrt(a) : a / G[k][k];
        }
      T w[6], q = T(0);
      for (int r = 0; r < np; ++r) {
        T a = chi[r] - th[r];
        for (int m = 0; m < r; ++m) a -= G[r][m] * w[m];
        w[r] = a / G[r][r];
        q += w[r] * w[r];
      }
      return -T(0.5) * q;
    }
    case M_BB1_FLUXNOISE1D: {
      // BB1 luminosity PDF, PAPER.md:256 (Eq. 5.1) = :423 (Eq. C.2), as a density in x = ln L (Jacobian L):
      //   L f(L) = C (L/u)^(beta+1) (1 - e^(-L/l)) e^(-L/u),   theta = (beta, ln l, ln u);
      // truncated to [x_lo, x_hi] (large L "formally excluded by truncation").
      if (!(chi[0] >= consts[C_XLO] && chi[0] <= consts[C_XHI])) return -std::numeric_limits<T>::infinity();
      const T Lum = std::exp(chi[0]), l = std::exp(th[1]), u = std::exp(th[2]);
      const T logC = (T)bb1_log_norm((double)th[0], (double)l, (double)u);
      return logC + (th[0] + T(1)) * (chi[0] - th[2]) + std::log(-std::expm1(-Lum / l)) - Lum / u;
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
    case M_NORMAL3D_KNOWNCOV: case M_NORMAL4D_KNOWNCOV: case M_NORMAL5D_KNOWNCOV: case M_NORMAL6D_KNOWNCOV:
      // "uniform hyperpriors", on a wide box so they are proper
      for (int j = 0; j < normal_family_p(model); ++j)
        if (!(std::fabs(th[j]) <= 1e3)) return ninf;
      return 0.0;
    case M_BB1_FLUXNOISE1D:
      // PAPER.md:277-290 (Eq. 5.3-5.5): truncated Cauchy in beta on (-2, 0), log-flat in u, flat in l on l < u
      // (p(l|u) = 1/u).  As a density in the sampled coordinates (beta, ln l, ln u) that is
      // l / (u (1 + beta^2)) -- Eq. 5.5 as printed (reading R17); box |ln l|, |ln u| <= 30 keeps it proper.
      if (!(th[0] > -2.0 && th[0] < 0.0 && th[1] < th[2] && std::fabs(th[1]) <= 30.0 && std::fabs(th[2]) <= 30.0))
        return ninf;
      return th[1] - th[2] - std::log(1.0 + th[0] * th[0]);
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
  // M4: eta(F) = Phi((F - F_th)/sigma(F)) with the flux-dependent sigma of Eq. 5.8 (Eq. 5.10).  eta does
  // not depend on theta, so the paper's 2-D cubature again factorises: G(x) is tabulated once.
  // Inner rule: 512-point Gauss-Legendre in q = ln r on [ln r_min, ln r_max] (h(r) dr = 3 e^(3q) dq/(rmax^3 - rmin^3));
  // the detection edge has a fixed width (1/(2 nu) ~ 0.1) in q wherever it falls, which a rule in r would not resolve
  // at small L.  selection_integral_2d() below is the same tensor-product rule written as the plain double sum.
  static double eta_bb1(double F, const double* c) {
    const double sg = std::sqrt(c[B_SIG0] * c[B_SIG0] + (c[B_ANOISE] * F) * (c[B_ANOISE] * F));
    return 0.5 * std::erfc(-((F - c[B_FTH]) / sg) / 1.4142135623730950488016887242097);
  }
  void build_bb1(const double* c) {
    const int NX = 1024, NQ = 512;
    const double four_pi = 12.566370614359172953850573533118;
    xk.assign(NX, 0.0); Wk.assign(NX, 0.0);
    std::vector<double> wx(NX), qj(NQ), wq(NQ);
    gauss_legendre(NX, c[C_XLO], c[C_XHI], xk.data(), wx.data());
    gauss_legendre(NQ, std::log(c[C_RMIN]), std::log(c[C_RMAX]), qj.data(), wq.data());
    const double vol = c[C_RMAX] * c[C_RMAX] * c[C_RMAX] - c[C_RMIN] * c[C_RMIN] * c[C_RMIN];
    for (int k = 0; k < NX; ++k) {
      long double G = 0.0L;
      for (int j = 0; j < NQ; ++j) {
        const double r = std::exp(qj[j]);
        const double F = std::exp(xk[k]) / (four_pi * r * r);
        G += (long double)(wq[j] * (3.0 * r * r * r / vol) * eta_bb1(F, c));
      }
      Wk[k] = wx[k] * (double)G;
    }
  }
  // I(theta) = int dx rho(x; theta) G(x), the denominator of Eq. 4.4; T(theta) = -N log I(theta) is the
  // theta-only term of log L = sum_i [log rho(x_i) + log l_i] - N log I   (Eq. 4.3 with mu = h rho / I).
  double bb1_integral(const double* th, const double* c) const {
    long double acc = 0.0L;
    double x[1], d[2] = {0.0, 0.0};
    for (size_t k = 0; k < xk.size(); ++k) {
      x[0] = xk[k];
      acc += (long double)(Wk[k] * std::exp(logpop<double>(M_BB1_FLUXNOISE1D, x, d, th, c)));
    }
    return (double)acc;
  }
  // the same integral as the plain 2-D tensor-product cubature, nothing tabulated (slow; pins the table route)
  static double selection_integral_2d(const double* th, const double* c) {
    const int NX = 1024, NQ = 512;
    const double four_pi = 12.566370614359172953850573533118;
    std::vector<double> xs(NX), wx(NX), qj(NQ), wq(NQ);
    gauss_legendre(NX, c[C_XLO], c[C_XHI], xs.data(), wx.data());
    gauss_legendre(NQ, std::log(c[C_RMIN]), std::log(c[C_RMAX]), qj.data(), wq.data());
    const double vol = c[C_RMAX] * c[C_RMAX] * c[C_RMAX] - c[C_RMIN] * c[C_RMIN] * c[C_RMIN];
    long double acc = 0.0L;
    double x[1], d[2] = {0.0, 0.0};
    for (int k = 0; k < NX; ++k) {
      x[0] = xs[k];
      const double rho = std::exp(logpop<double>(M_BB1_FLUXNOISE1D, x, d, th, c));
      for (int j = 0; j < NQ; ++j) {
        const double r = std::exp(qj[j]);
        const double F = std::exp(xs[k]) / (four_pi * r * r);
        acc += (long double)(wx[k] * wq[j] * rho * (3.0 * r * r * r / vol) * eta_bb1(F, c));
      }
    }
    return (double)acc;
  }
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
