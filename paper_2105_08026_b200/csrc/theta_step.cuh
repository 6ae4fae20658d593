// theta_step.cuh -- the theta Metropolis-Hastings tail (PAPER.md:108 Eq. 2.5, :142), host + device.
//
// The same two functions run (a) on thread 0 of every block of the persistent kernel, redundantly and
// bit-identically (THETA_DEVICE_TAIL), (b) in the 1-block tail kernel (THETA_GRAPH, debug_step), and
// (c) on the host (THETA_HOST, the paper's own split).  DESIGN.md section 8.3.
#pragma once
#include "models.cuh"

namespace hm {

constexpr int MAXD = 8;                       // max dtheta
constexpr int MAXTRI = MAXD * (MAXD + 1) / 2;
constexpr int NPART = 5;                      // per-block partials: S, Delta, Tq, n_accept, n_nonfinite

// Iteration state: lives in global memory between launches, in shared memory inside the persistent kernel.
struct Iter {
  double theta[MAXD], thetaP[MAXD];   // theta and the pre-drawn proposal theta' of iteration t
  double Lth[MAXTRI];                 // packed lower-triangular proposal factor of the theta RAM
  double z[MAXD];                     // z_theta of iteration t (needed again by the RAM update)
  ThetaK kc, kp;                      // theta-derived constants at theta / theta'
  double T_cur, lp_cur, lp_prop;      // theta-only term and log prior at theta; log prior at theta'
  double eta;                         // eta_n of iteration t, n = t + 1
  // taps of the last decision (debug_step / host mode read them)
  double S, Delta, T_prop, log_r, alpha_theta, u_theta, T_cur_used, lp_cur_used;
  long long t;                        // the PREPARED iteration (1-based): t-1 iterations are complete
  long long mom_count, trace_rows;
  unsigned long long chi_acc, theta_acc, theta_prop_n, nonfinite;
  int accepted_theta, trace_write;
};

struct TailCfg {
  int model, dtheta, freeze_theta, keep_moments;
  unsigned long long seed;
  double astar_theta, eta_exp;
  long long burn_in, max_trace_rows;
  int thin, pad_;
};

HM_HD int tri(int r, int c) { return r * (r + 1) / 2 + c; }

// RAM step 3 (Eq. 2.6) for general p as a rank-one update in closed form:
//   chol(I + c u u^T) = K,  K_jj = sqrt(s_{j+1}/s_j),  K_ij = c u_i u_j / sqrt(s_j s_{j+1}) (i > j),
//   s_j = 1 + c sum_{k<j} u_k^2;  then L <- L K, which is lower-triangular with positive diagonal and
//   satisfies (L K)(L K)^T = L (I + c u u^T) L^T, hence is THE left Cholesky factor.
//   1 + c >= 1 - alpha_* > 0, so every s_j > 0.
HM_HD void ram_update_general(int p, double* L, const double* z, double c) {
  double n2 = 0.0;
  for (int j = 0; j < p; ++j) n2 += z[j] * z[j];
  const double rn = 1.0 / sqrt(n2);
  double u[MAXD], rs[MAXD + 1], Kd[MAXD], g[MAXD];
  double s = 1.0;
  rs[0] = 1.0;
  for (int j = 0; j < p; ++j) { u[j] = z[j] * rn; s += c * u[j] * u[j]; rs[j + 1] = sqrt(s); }
  for (int j = 0; j < p; ++j) { Kd[j] = rs[j + 1] / rs[j]; g[j] = c * u[j] / (rs[j] * rs[j + 1]); }
  for (int i = 0; i < p; ++i) {
    double w = 0.0;                               // sum_{k=j+1..i} L_ik u_k
    for (int j = i; j >= 0; --j) {
      const double lij = L[tri(i, j)];
      L[tri(i, j)] = lij * Kd[j] + g[j] * w;
      w += lij * u[j];
    }
  }
}

// Everything about iteration t that does not depend on the sweep: eta_n, the theta proposal
// theta' = theta + L_theta z (drawn BEFORE the sweep so one pass evaluates f at theta and theta'), its
// derived constants and prior.
HM_HD void prepare_iteration(Iter& it, const TailCfg& c, long long t) {
  it.t = t;
  it.eta = pow((double)(t + 1), -c.eta_exp);                 // RAM iteration n = t + 1 (X_1, S_1 are initial values)
  if (!c.freeze_theta) {
    normals(c.seed, KIND_THETA, 0ull, (uint32_t)t, c.dtheta, it.z);
    for (int r = 0; r < c.dtheta; ++r) {
      double s = it.theta[r];
      for (int k = 0; k <= r; ++k) s += it.Lth[tri(r, k)] * it.z[k];
      it.thetaP[r] = s;
    }
    it.kp = theta_consts(c.model, it.thetaP);
    it.lp_prop = log_prior(c.model, it.thetaP);
  } else {
    for (int r = 0; r < c.dtheta; ++r) it.thetaP[r] = it.theta[r];
    it.kp = it.kc;
    it.lp_prop = it.lp_cur;
  }
}

// The theta decision of iteration it.t from the reduced sweep totals tot[NPART] = {S, Delta, Tq, nacc, nnan}.
// Sets it.trace_write when the (new) theta has to be appended to the thinned trace at row it.trace_rows - 1.
HM_HD void tail_decide(Iter& it, const TailCfg& c, const double* tot) {
  it.S = tot[0];
  it.Delta = tot[1];
  it.chi_acc += (unsigned long long)tot[3];
  it.nonfinite += (unsigned long long)tot[4];
  it.accepted_theta = 0;
  it.T_prop = 0.0; it.log_r = 0.0; it.alpha_theta = 0.0; it.u_theta = 0.0;
  it.T_cur_used = it.T_cur; it.lp_cur_used = it.lp_cur;
  if (!c.freeze_theta) {
    double la;
    if (it.lp_prop == -INFINITY) {
      it.log_r = -INFINITY; la = -INFINITY;
    } else {
      // M1: T(theta') = -A' sum_k W_k phi(x_k; theta') -- minus the expected detected count (Eq. 4.4 denominator)
      it.T_prop = (c.model == M_THINNED_SCHECHTER1D) ? -exp(it.kp.v[2]) * tot[2] : 0.0;
      it.log_r = it.Delta + (it.T_prop - it.T_cur) + (it.lp_prop - it.lp_cur);
      la = (it.log_r != it.log_r) ? -INFINITY : fmin(0.0, it.log_r);
    }
    it.alpha_theta = exp(la);
    const U4 r = stream(c.seed, KIND_THETA, 0ull, (uint32_t)it.t, 0u);
    it.u_theta = u01(r.x, r.y);
    it.theta_prop_n += 1;
    if (it.u_theta < it.alpha_theta) {
      it.accepted_theta = 1;
      it.theta_acc += 1;
      for (int r2 = 0; r2 < c.dtheta; ++r2) it.theta[r2] = it.thetaP[r2];
      it.kc = it.kp; it.T_cur = it.T_prop; it.lp_cur = it.lp_prop;
    }
    ram_update_general(c.dtheta, it.Lth, it.z, it.eta * (it.alpha_theta - c.astar_theta));
  }
  if (c.keep_moments && it.t > c.burn_in) it.mom_count += 1;
  it.trace_write = 0;
  if (it.t > c.burn_in && ((it.t - c.burn_in) % c.thin) == 0 && it.trace_rows < c.max_trace_rows) {
    it.trace_rows += 1;
    it.trace_write = 1;
  }
}

}  // namespace hm
