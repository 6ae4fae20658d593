// models.cuh -- compiled-in models of the CUDA path: the counterpart of the paper's two user functions
// (member log-likelihood log l_i(chi); population log-density log f(chi; theta), PAPER.md:80;
// see PAPER.md:144, :391) plus the theta prior.  Definitions: DESIGN.md section 3.
//
// Layout choices made for the kernels (not part of the model):
//   - every theta-only transcendental (exp(-2 lambda), exp(-x*), log cosh zeta ...) is hoisted into a small
//     table ThetaK computed once per iteration by the theta tail, for theta and for theta';
//   - Gaussian error columns are stored as h = 1/(2 sigma^2) so the sweep has no division;
//   - M1 evaluates e^chi once per point and shares it between the flux likelihood and the population term.
#pragma once
#include <cmath>
#include <cstdint>
#include "philox.cuh"
#include "fastmath.cuh"

namespace hm {

enum : int { M_NORMAL1D = 0, M_THINNED_SCHECHTER1D = 1, M_BINORMAL2D = 2, M_LINREG_ME1D = 3, M_BB1_FLUXNOISE1D = 4,
             M_NORMAL3D_KNOWNCOV = 5, M_NORMAL4D_KNOWNCOV = 6, M_NORMAL5D_KNOWNCOV = 7, M_NORMAL6D_KNOWNCOV = 8 };
// latent dimension of the normal-normal family (PAPER.md:146-166 for p = 3; Eq. 2.6 holds for any p), 0 for the others
HM_HD constexpr int normal_family_p(int model) {
  return (model >= M_NORMAL3D_KNOWNCOV && model <= M_NORMAL6D_KNOWNCOV) ? model - M_NORMAL3D_KNOWNCOV + 3 : 0;
}
enum : int { MC_FLIM = 0, MC_SIGF = 1, MC_XLO = 2, MC_XHI = 3, MC_RMIN = 4, MC_RMAX = 5, MC_INV2S2 = 6 };
// M4 keeps sigma_0^2 and alpha^2 (Eq. 5.8) where M1 keeps F_lim and sigma_F; the threshold goes to slot 6
enum : int { MB_S0SQ = 0, MB_A2 = 1, MB_FTH = 6 };
// normal-normal family (p = 3 .. 6): h_j = 1/(2 sigma_j^2) (p values), then Q = the packed lower triangle of C_pop^-1 with
// the diagonal halved (p (p + 1) / 2 values, starting at slot p), so that -1/2 e^T C_pop^-1 e = -sum_i e_i sum_{j<=i} Q_ij e_j
enum : int { MN_H = 0 };
constexpr int MC_N = 27;      // model-constant slots (p = 6: 6 + 21)
constexpr int NQUAD = 1024;   // selection-integral nodes (BASELINE.json configs[1])

template <int MODEL> struct ModelDims;
template <> struct ModelDims<M_NORMAL1D>            { static constexpr int p = 1, dtheta = 2, ncols = 2, nconsts = 0; };
template <> struct ModelDims<M_THINNED_SCHECHTER1D> { static constexpr int p = 1, dtheta = 3, ncols = 2, nconsts = 6; };
template <> struct ModelDims<M_BINORMAL2D>          { static constexpr int p = 2, dtheta = 5, ncols = 4, nconsts = 0; };
template <> struct ModelDims<M_LINREG_ME1D>         { static constexpr int p = 1, dtheta = 3, ncols = 3, nconsts = 0; };
template <> struct ModelDims<M_BB1_FLUXNOISE1D>     { static constexpr int p = 1, dtheta = 3, ncols = 2, nconsts = 7; };
template <> struct ModelDims<M_NORMAL3D_KNOWNCOV>   { static constexpr int p = 3, dtheta = 3, ncols = 3, nconsts = 9; };
template <> struct ModelDims<M_NORMAL4D_KNOWNCOV>   { static constexpr int p = 4, dtheta = 4, ncols = 4, nconsts = 14; };
template <> struct ModelDims<M_NORMAL5D_KNOWNCOV>   { static constexpr int p = 5, dtheta = 5, ncols = 5, nconsts = 20; };
template <> struct ModelDims<M_NORMAL6D_KNOWNCOV>   { static constexpr int p = 6, dtheta = 6, ncols = 6, nconsts = 27; };

// models whose likelihood carries a theta-only selection term (the denominator of Eq. 4.4) summed over
// the NQUAD nodes, whose latent is x = ln L with flux columns (Fhat, g = 1/(4 pi r^2)) and a bounded support
HM_HD constexpr bool has_selection(int model) { return model == M_THINNED_SCHECHTER1D || model == M_BB1_FLUXNOISE1D; }

inline bool model_dims(int model, int* p, int* dtheta, int* ncols, int* nconsts) {
  switch (model) {
    case M_NORMAL1D:            *p = 1; *dtheta = 2; *ncols = 2; *nconsts = 0; return true;
    case M_THINNED_SCHECHTER1D: *p = 1; *dtheta = 3; *ncols = 2; *nconsts = 6; return true;
    case M_BINORMAL2D:          *p = 2; *dtheta = 5; *ncols = 4; *nconsts = 0; return true;
    case M_LINREG_ME1D:         *p = 1; *dtheta = 3; *ncols = 3; *nconsts = 0; return true;
    case M_BB1_FLUXNOISE1D:     *p = 1; *dtheta = 3; *ncols = 2; *nconsts = 7; return true;
    case M_NORMAL3D_KNOWNCOV: case M_NORMAL4D_KNOWNCOV: case M_NORMAL5D_KNOWNCOV: case M_NORMAL6D_KNOWNCOV: {
      const int np = normal_family_p(model);
      *p = np; *dtheta = np; *ncols = np; *nconsts = np + np * (np + 1) / 2; return true;
    }
  }
  return false;
}

// theta-derived constants, fp64
struct ThetaK { double v[8]; };

// theta_consts in three independent parts (disjoint entries of k) so that the block-parallel tail can give each
// part to its own warp; part 0 carries the bulk, parts 1 and 2 only exist for M2's cosh/log and tanh.
HM_HD void theta_consts_part(int model, int part, const double* th, ThetaK& k) {
  switch (model) {
    case M_NORMAL1D:            // (mu, lambda): f = -lambda - (chi - mu)^2 * [e^(-2 lambda)/2]
      if (part == 0) { k.v[0] = th[0]; k.v[1] = th[1]; k.v[2] = 0.5 * hm_exp_any(-2.0 * th[1]); }
      break;
    case M_LINREG_ME1D:         // (a, b, lambda): f = -lambda - (chi - a - b z)^2 * [e^(-2 lambda)/2]
      if (part == 0) { k.v[0] = th[0]; k.v[1] = th[1]; k.v[2] = th[2]; k.v[3] = 0.5 * hm_exp_any(-2.0 * th[2]); }
      break;
    case M_THINNED_SCHECHTER1D: // (alpha, x*, a): f = a + (alpha+1)(chi - x*) - e^chi e^(-x*);  v[4] = A = e^a
      if (part == 0) { k.v[0] = th[0] + 1.0; k.v[1] = th[1]; k.v[2] = th[2]; k.v[3] = hm_exp_any(-th[1]); }
      if (part == 1) k.v[4] = hm_exp_any(th[2]);
      break;
    case M_BINORMAL2D:          // (m1, m2, l1, l2, zeta): f = c0 - h (u1^2 - 2 rho u1 u2 + u2^2)
      if (part == 0) { k.v[0] = th[0]; k.v[1] = th[1]; k.v[2] = hm_exp_any(-th[2]); k.v[3] = hm_exp_any(-th[3]); }
      if (part == 1) { const double ch = cosh(th[4]); k.v[4] = -th[2] - th[3] + log(ch); k.v[5] = 0.5 * ch * ch; }
      if (part == 2) k.v[6] = tanh(th[4]);
      break;
    case M_NORMAL3D_KNOWNCOV: case M_NORMAL4D_KNOWNCOV: case M_NORMAL5D_KNOWNCOV: case M_NORMAL6D_KNOWNCOV:
      // theta = mu; C_pop is a known model constant
      if (part == 0) { k.v[0] = th[0]; k.v[1] = th[1]; k.v[2] = th[2]; if (model >= M_NORMAL4D_KNOWNCOV) k.v[3] = th[3]; if (model >= M_NORMAL5D_KNOWNCOV) k.v[4] = th[4]; if (model >= M_NORMAL6D_KNOWNCOV) k.v[5] = th[5]; }
      break;
    case M_BB1_FLUXNOISE1D:
      // (beta, ln l, ln u): f = log C + (beta+1)(x - ln u) + log(1 - e^(-L/l)) - L/u   (Eq. 5.1 in x = ln L).
      // The normaliser C(beta, u, l) of Eq. C.3 multiplies both rho(x_i; theta) and the selection integral I(theta) of
      // Eq. 4.4, so it cancels in mu = h rho / I and in every Metropolis ratio: the device works with the SHAPE
      // rho/C throughout (no lgamma / expm1 / log1p chain on the critical path of the theta step) and the taps of
      // cudahm_debug_step add log C back on the host (cudahm.cu::bb1_log_norm), so they read in the paper's convention.
      if (part == 0) { k.v[0] = th[0] + 1.0; k.v[1] = th[2]; k.v[3] = hm_exp_any(-th[1]); k.v[4] = hm_exp_any(-th[2]); }
      break;
  }
}

// theta-only term T(theta) from the node sum  sum_k W_k rho(x_k; theta):
//   M1: minus the expected detected count, -A sum;   M4: -N log sum  (Eq. 4.3 with mu = h rho / I, Eq. 4.4; rho/C)
HM_HD double theta_only_from_sum(int model, const ThetaK& k, double tq, double n_objects) {
  if (model == M_THINNED_SCHECHTER1D) return -k.v[4] * tq;
#ifdef __CUDA_ARCH__
  if (model == M_BB1_FLUXNOISE1D) return -n_objects * hm_log_pos(tq);
#else
  if (model == M_BB1_FLUXNOISE1D) return -n_objects * std::log(tq);
#endif
  return 0.0;
}

HM_HD ThetaK theta_consts(int model, const double* th) {
  ThetaK k;
#pragma unroll
  for (int j = 0; j < 8; ++j) k.v[j] = 0.0;
  for (int part = 0; part < 3; ++part) theta_consts_part(model, part, th, k);
  return k;
}

// log prior: flat on a wide box; M1 slope: truncated Cauchy of Eq. 5.4
HM_HD double log_prior(int model, const double* th) {
  const double ninf = -INFINITY;
  switch (model) {
    case M_NORMAL1D:
      return (fabs(th[0]) <= 1e3 && fabs(th[1]) <= 10.0) ? 0.0 : ninf;
    case M_LINREG_ME1D:
      return (fabs(th[0]) <= 1e3 && fabs(th[1]) <= 1e3 && fabs(th[2]) <= 10.0) ? 0.0 : ninf;
    case M_BINORMAL2D:
      return (fabs(th[0]) <= 1e3 && fabs(th[1]) <= 1e3 && fabs(th[2]) <= 10.0 && fabs(th[3]) <= 10.0 &&
              fabs(th[4]) <= 10.0) ? 0.0 : ninf;
    case M_THINNED_SCHECHTER1D:
      return (th[0] > -2.0 && th[0] < 0.0 && fabs(th[1]) <= 20.0 && fabs(th[2]) <= 50.0)
                 ? -hm_log_any_pos(1.0 + th[0] * th[0]) : ninf;
    case M_NORMAL3D_KNOWNCOV: case M_NORMAL4D_KNOWNCOV: case M_NORMAL5D_KNOWNCOV: case M_NORMAL6D_KNOWNCOV: {
      // "uniform hyperpriors" on a wide box
      bool in = fabs(th[0]) <= 1e3 && fabs(th[1]) <= 1e3 && fabs(th[2]) <= 1e3;
      if (model >= M_NORMAL4D_KNOWNCOV) in = in && fabs(th[3]) <= 1e3;
      if (model >= M_NORMAL5D_KNOWNCOV) in = in && fabs(th[4]) <= 1e3;
      if (model >= M_NORMAL6D_KNOWNCOV) in = in && fabs(th[5]) <= 1e3;
      return in ? 0.0 : ninf;
    }
    case M_BB1_FLUXNOISE1D:     // Eq. 5.5 as a density in (beta, ln l, ln u): l / (u (1 + beta^2)), l < u
      return (th[0] > -2.0 && th[0] < 0.0 && th[1] < th[2] && fabs(th[1]) <= 30.0 && fabs(th[2]) <= 30.0)
                 ? th[1] - th[2] - hm_log_any_pos(1.0 + th[0] * th[0]) : ninf;
  }
  return ninf;
}

// ---------------------------------------------------------------------------------------------------
// Plate-side evaluation.  T = state precision.  D = stored data columns of the object (h = 1/(2 sigma^2)).
// K<T> = ThetaK narrowed to T.  A "point" caches what the target and the population terms share.
template <class T> struct KT { T v[7]; };
template <class T> HM_HD KT<T> narrow(const ThetaK& k) {
  KT<T> r;
#pragma unroll
  for (int j = 0; j < 7; ++j) r.v[j] = (T)k.v[j];
  return r;
}

// e^x of the sweep: specialised version (fastmath.cuh); exp(-inf) = 0 is selected explicitly (alpha of a proposal
// outside the support)
__device__ __forceinline__ double hm_exp(double x) { const double r = hm_exp_fast(x); return x < -708.0 ? 0.0 : r; }
// alpha = e^la for la <= 0 (or -inf): one compare serves the clamp and the exact zero
__device__ __forceinline__ double hm_exp_nonpos(double la) {
  const bool tiny = la < -708.0;
  const double r = hm_exp_core(tiny ? -708.0 : la);
  return tiny ? 0.0 : r;
}
__device__ __forceinline__ float hm_exp_nonpos(float la) { return expf(la); }
// e^x of a model point whose target is -inf outside a bounded support: no argument check at all
__device__ __forceinline__ double hm_exp_point(double x) { return hm_exp_core(x); }
__device__ __forceinline__ float hm_exp_point(float x) { return expf(x); }
__device__ __forceinline__ float hm_exp(float x) { return expf(x); }

template <int MODEL, class T> struct Plate;

template <class T> struct Plate<M_NORMAL1D, T> {
  struct Pt { T x; };
  __device__ __forceinline__ static Pt point(const T* chi) { return Pt{chi[0]}; }
  // log l_i + log f(.; theta)
  __device__ __forceinline__ static T target(const Pt& q, const T* d, const KT<T>& k, const T*) {
    const T r = d[0] - q.x, s = q.x - k.v[0];
    return -(r * r) * d[1] - k.v[1] - (s * s) * k.v[2];
  }
  __device__ __forceinline__ static double pop(const Pt& q, const T*, const ThetaK& k, const double*) {
    const double s = (double)q.x - k.v[0];
    return -k.v[1] - (s * s) * k.v[2];
  }
};

template <class T> struct Plate<M_LINREG_ME1D, T> {
  struct Pt { T x; };
  __device__ __forceinline__ static Pt point(const T* chi) { return Pt{chi[0]}; }
  __device__ __forceinline__ static T target(const Pt& q, const T* d, const KT<T>& k, const T*) {
    const T r = d[0] - q.x, s = q.x - k.v[0] - k.v[1] * d[2];
    return -(r * r) * d[1] - k.v[2] - (s * s) * k.v[3];
  }
  __device__ __forceinline__ static double pop(const Pt& q, const T* d, const ThetaK& k, const double*) {
    const double s = (double)q.x - k.v[0] - k.v[1] * (double)d[2];
    return -k.v[2] - (s * s) * k.v[3];
  }
};

template <class T> struct Plate<M_THINNED_SCHECHTER1D, T> {
  struct Pt { T x, ex; };
  __device__ __forceinline__ static Pt point(const T* chi) { return Pt{chi[0], hm_exp_point(chi[0])}; }
  // mc = {F_lim, sigma_F, x_lo, x_hi, r_min, r_max, 1/(2 sigma_F^2)} narrowed to T
  __device__ __forceinline__ static T target(const Pt& q, const T* d, const KT<T>& k, const T* mc) {
    if (!(q.x >= mc[MC_XLO] && q.x <= mc[MC_XHI])) return -INFINITY;
    const T r = d[0] - d[1] * q.ex;
    return -(r * r) * mc[MC_INV2S2] + k.v[2] + k.v[0] * (q.x - k.v[1]) - q.ex * k.v[3];
  }
  __device__ __forceinline__ static double pop(const Pt& q, const T*, const ThetaK& k, const double*) {
    return k.v[2] + k.v[0] * ((double)q.x - k.v[1]) - (double)q.ex * k.v[3];
  }
};

// 1 - e^(-t), t >= 0, with full relative accuracy at small t (L << l)
__device__ __forceinline__ double hm_one_minus_exp_neg(double t) { return -hm_expm1_nonpos(-t); }
__device__ __forceinline__ float hm_one_minus_exp_neg(float t) { return -expm1f(-t); }
// 1/a for positive normal a: MUFU seed + two Newton steps (~1 ulp)
__device__ __forceinline__ double hm_rcp_pos(double a) {
  double r = hm_rcp_seed(a);
  double e = hm_fma(-a, r, 1.0);
  r = hm_fma(r, e, r);
  e = hm_fma(-a, r, 1.0);
  r = hm_fma(r, e, r);
  e = hm_fma(-a, r, 1.0);
  return hm_fma(r, e, r);
}
__device__ __forceinline__ float hm_rcp_pos(float a) { return 1.0f / a; }
__device__ __forceinline__ double hm_log_point(double x) { return hm_log_pos(x); }
__device__ __forceinline__ float hm_log_point(float x) { return logf(x); }

// M4, the paper's case study: BB1 population in x = ln L, member likelihood = the sampling density
// of Fhat as a function of F with sigma(F)^2 = sigma_0^2 + (alpha F)^2 (Eq. 5.6, 5.8).
template <class T> struct Plate<M_BB1_FLUXNOISE1D, T> {
  struct Pt { T x, ex; };
  __device__ __forceinline__ static Pt point(const T* chi) { return Pt{chi[0], hm_exp_point(chi[0])}; }
  // mc = {sigma_0^2, alpha^2, x_lo, x_hi, r_min, r_max, F_th} narrowed to T
  __device__ __forceinline__ static T target(const Pt& q, const T* d, const KT<T>& k, const T* mc) {
    if (!(q.x >= mc[MC_XLO] && q.x <= mc[MC_XHI])) return -INFINITY;
    const T F = d[1] * q.ex, r = d[0] - F;
    const T inv = hm_rcp_pos(mc[MB_S0SQ] + mc[MB_A2] * F * F);          // 1/sigma(F)^2
    const T w = hm_one_minus_exp_neg(q.ex * k.v[3]);                     // 1 - e^(-L/l)
    const T c0 = -k.v[0] * k.v[1];
    // -log sigma(F) + log(1 - e^(-L/l)) in one logarithm
    return T(0.5) * hm_log_point(w * w * inv) - T(0.5) * (r * r) * inv + c0 + k.v[0] * q.x - q.ex * k.v[4];
  }
  __device__ __forceinline__ static double pop(const Pt& q, const T*, const ThetaK& k, const double*) {
    const double c0 = -k.v[0] * k.v[1];
    return c0 + k.v[0] * (double)q.x + hm_log_pos(hm_one_minus_exp_neg((double)q.ex * k.v[3])) - (double)q.ex * k.v[4];
  }
};

// The normal-normal family (PAPER.md:146-166 is p = 3): chi ~ N_p(mu, C_pop), y_j ~ N(chi_j, sigma_j^2), C_pop and sigma_j known.
template <int P, class T> struct PlateNormalP {
  struct Pt { T x[P]; };
  __device__ __forceinline__ static Pt point(const T* chi) {
    Pt q;
#pragma unroll
    for (int j = 0; j < P; ++j) q.x[j] = chi[j];
    return q;
  }
  // sum_i e_i sum_{j<=i} Q_ij e_j with Q the packed lower triangle (diagonal halved)
  template <class R>
  __device__ __forceinline__ static R quad(const R* e, const R* Q) {
    R s = R(0);
#pragma unroll
    for (int i = 0; i < P; ++i) {
      R a = R(0);
#pragma unroll
      for (int j = 0; j <= i; ++j) a += Q[i * (i + 1) / 2 + j] * e[j];
      s += e[i] * a;
    }
    return s;
  }
  __device__ __forceinline__ static T target(const Pt& q, const T* d, const KT<T>& k, const T* mc) {
    T s = T(0), e[P];
#pragma unroll
    for (int j = 0; j < P; ++j) { const T r = d[j] - q.x[j]; s -= (r * r) * mc[MN_H + j]; e[j] = q.x[j] - k.v[j]; }
    return s - quad<T>(e, mc + P);
  }
  __device__ __forceinline__ static double pop(const Pt& q, const T*, const ThetaK& k, const double* mc) {
    double e[P];
#pragma unroll
    for (int j = 0; j < P; ++j) e[j] = (double)q.x[j] - k.v[j];
    return -quad<double>(e, mc + P);
  }
};
template <class T> struct Plate<M_NORMAL3D_KNOWNCOV, T> : PlateNormalP<3, T> {};
template <class T> struct Plate<M_NORMAL4D_KNOWNCOV, T> : PlateNormalP<4, T> {};
template <class T> struct Plate<M_NORMAL5D_KNOWNCOV, T> : PlateNormalP<5, T> {};
template <class T> struct Plate<M_NORMAL6D_KNOWNCOV, T> : PlateNormalP<6, T> {};

// one node of the selection sum: W_k rho(x_k; theta) from the node's x_k and e^(x_k)
template <int MODEL>
__device__ __forceinline__ double selection_term(const ThetaK& k, double W, double x, double ex) {
  if (MODEL == M_THINNED_SCHECHTER1D) return W * hm_exp(k.v[0] * (x - k.v[1]) - ex * k.v[3]);
  if (MODEL == M_BB1_FLUXNOISE1D) {
    return W * hm_exp(k.v[0] * (x - k.v[1]) - ex * k.v[4]) * hm_one_minus_exp_neg(ex * k.v[3]);
  }
  return 0.0;
}
__device__ __forceinline__ double selection_term_rt(int model, const ThetaK& k, double W, double x, double ex) {
  return model == M_THINNED_SCHECHTER1D ? selection_term<M_THINNED_SCHECHTER1D>(k, W, x, ex)
                                        : selection_term<M_BB1_FLUXNOISE1D>(k, W, x, ex);
}

template <class T> struct Plate<M_BINORMAL2D, T> {
  struct Pt { T x1, x2; };
  __device__ __forceinline__ static Pt point(const T* chi) { return Pt{chi[0], chi[1]}; }
  __device__ __forceinline__ static T target(const Pt& q, const T* d, const KT<T>& k, const T*) {
    const T r1 = d[0] - q.x1, r2 = d[1] - q.x2;
    const T u1 = (q.x1 - k.v[0]) * k.v[2], u2 = (q.x2 - k.v[1]) * k.v[3];
    return -(r1 * r1) * d[2] - (r2 * r2) * d[3] + k.v[4] - k.v[5] * (u1 * u1 - T(2) * k.v[6] * u1 * u2 + u2 * u2);
  }
  __device__ __forceinline__ static double pop(const Pt& q, const T*, const ThetaK& k, const double*) {
    const double u1 = ((double)q.x1 - k.v[0]) * k.v[2], u2 = ((double)q.x2 - k.v[1]) * k.v[3];
    return k.v[4] - k.v[5] * (u1 * u1 - 2.0 * k.v[6] * u1 * u2 + u2 * u2);
  }
};

}  // namespace hm
