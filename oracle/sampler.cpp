// oracle/sampler.cpp -- single-threaded Metropolis-within-Gibbs oracle.  TEST INFRASTRUCTURE ONLY.
//
// Follows the paper step by step, in its order and notation:
//   Gibbs cycle   psi_i ~ p(psi_i | theta, D_i) for all i, then theta ~ p(theta | psi)
//   RAM           1. Y = X + S U   2. accept w.p. alpha = min{1, pi(Y)/pi(X)}
//                 3. S_n S_n^T = S (I + eta_n (alpha_n - alpha_*) U U^T/||U||^2) S^T,
//                    S_n = the left Cholesky factor of the right-hand side
//   theta step    Metropolis-Hastings using sum_i log f(chi_i; theta') (+ prior, + T)
// No blocking, fusion or reordering: objects are visited in index order, the update matrix is formed
// and factored in full, sums run in index order in long double.  Readings of silent points: DESIGN.md 6.
// Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC (oracle/build.py).
#include "oracle.h"
#include "models.hpp"
#include "rng.hpp"

#include <algorithm>
#include <cstring>
#include <memory>
#include <vector>

namespace oracle {

static inline int ntri(int p) { return p * (p + 1) / 2; }
static inline int tri(int r, int c) { return r * (r + 1) / 2 + c; }   // packed lower triangle, row-major

// Step 3 of RAM, plain definition: form M = S (I + c u u^T) S^T with u = z/||z||, then factor M.
template <class T>
static void ram_update(int p, const T* L, const T* z, T c, T* out) {
  T S[8][8] = {}, A[8][8] = {}, SA[8][8] = {}, M[8][8] = {}, C[8][8] = {};
  T nrm2 = 0;
  for (int j = 0; j < p; ++j) nrm2 += z[j] * z[j];
  const T nrm = std::sqrt(nrm2);
  T u[8];
  for (int j = 0; j < p; ++j) u[j] = z[j] / nrm;
  for (int r = 0; r < p; ++r)
    for (int k = 0; k <= r; ++k) S[r][k] = L[tri(r, k)];
  for (int r = 0; r < p; ++r)
    for (int k = 0; k < p; ++k) A[r][k] = (r == k ? T(1) : T(0)) + c * u[r] * u[k];
  for (int r = 0; r < p; ++r)
    for (int k = 0; k < p; ++k) { T s = 0; for (int m = 0; m < p; ++m) s += S[r][m] * A[m][k]; SA[r][k] = s; }
  for (int r = 0; r < p; ++r)
    for (int k = 0; k < p; ++k) { T s = 0; for (int m = 0; m < p; ++m) s += SA[r][m] * S[k][m]; M[r][k] = s; }
  // Cholesky-Banachiewicz: M = C C^T, C lower-triangular with positive diagonal
  for (int r = 0; r < p; ++r)
    for (int k = 0; k <= r; ++k) {
      T s = M[r][k];
      for (int m = 0; m < k; ++m) s -= C[r][m] * C[k][m];
      C[r][k] = (r == k) ? std::sqrt(s) : s / C[k][k];
    }
  for (int r = 0; r < p; ++r)
    for (int k = 0; k <= r; ++k) out[tri(r, k)] = C[r][k];
}

struct Base {
  virtual ~Base() {}
  oracle_config cfg{};
  Dims dims{};
  bool have_data = false, have_init = false, have_consts = false;
  int64_t t = 0;                     // Gibbs iterations done
  std::vector<double> theta, Ltheta; // fp64 always
  std::vector<double> consts;
  SelectionTable table;
  std::vector<double> trace;         // rows of dtheta
  std::vector<double> mom_mean, mom_M2;
  int64_t mom_count = 0;
  std::vector<uint8_t> mask;         // empty = every object is updated (held-fixed members)
  std::vector<uint32_t> counters;    // RAM updates each object has taken so far
  int64_t n_active() const {
    if (mask.empty()) return cfg.n_objects;
    int64_t k = 0;
    for (uint8_t m : mask) k += m ? 1 : 0;
    return k;
  }
  oracle_stats stats{};
  virtual int set_data(const double* const* cols, int n_cols) = 0;
  virtual int set_init(const double* chi0, const double* theta0, const double* chol0) = 0;
  virtual int step(int64_t burn_in, int32_t thin, oracle_taps* taps) = 0;
  virtual int sweep_part(int64_t burn_in, oracle_taps* taps, double* tot) = 0;
  virtual int decide_part(int64_t burn_in, int32_t thin, oracle_taps* taps, const double* tot) = 0;
  virtual int get_state(double* chi, double* L, double* th, double* Lth, int64_t* tt) = 0;
  virtual int set_state(const double* chi, const double* L, const double* th, const double* Lth, int64_t tt) = 0;
  // user prior on theta ("To override this default prior ..."): independent normal factors
  double user_prior(const double* th) const {
    double s = 0.0;
    for (int j = 0; j < dims.dtheta; ++j) {
      const double r = (th[j] - cfg.prior_mean[j]) * cfg.prior_isd[j];
      s += -0.5 * r * r;
    }
    return s;
  }
  double theta_only(const double* th) const {
    if (cfg.model == M_THINNED_SCHECHTER1D) return table.theta_only(th);
    // M4: log L = sum_i [log rho(x_i; theta) + log l_i(x_i)] - N log I(theta)   (Eq. 4.3-4.4)
    if (cfg.model == M_BB1_FLUXNOISE1D)
      return -(double)(cfg.n_objects_total ? cfg.n_objects_total : cfg.n_objects) * std::log(table.bb1_integral(th, consts.data()));
    return 0.0;
  }
};

template <class T>
struct Impl : Base {
  std::vector<T> chi, L, data, consts_T;   // SoA: [component][object]

  int set_data(const double* const* cols, int n_cols) override {
    if (n_cols != dims.n_cols) return ORACLE_E_INVALID;
    const int64_t N = cfg.n_objects;
    data.resize((size_t)dims.n_cols * N);
    for (int c = 0; c < n_cols; ++c)
      for (int64_t i = 0; i < N; ++i) data[(size_t)c * N + i] = (T)cols[c][i];
    have_data = true;
    return ORACLE_OK;
  }

  int set_init(const double* chi0, const double* theta0, const double* chol0) override {
    if (!have_data || (dims.n_consts > 0 && !have_consts)) return ORACLE_E_STATE;
    const int64_t N = cfg.n_objects;
    const int p = dims.p, dt = dims.dtheta;
    chi.assign((size_t)p * N, T(0));
    L.assign((size_t)ntri(p) * N, T(0));
    for (int64_t i = 0; i < N; ++i) {
      if (chi0) {
        for (int j = 0; j < p; ++j) chi[(size_t)j * N + i] = (T)chi0[(size_t)j * N + i];
      } else if (cfg.model == M_THINNED_SCHECHTER1D || cfg.model == M_BB1_FLUXNOISE1D) {
        // X_1 with pi(X_1) > 0: the flux estimate inverted, clamped to the support
        double x = std::log((double)data[i] / (double)data[(size_t)N + i]);
        x = std::min(std::max(x, consts[C_XLO]), consts[C_XHI]);
        chi[i] = (T)x;
      } else {
        for (int j = 0; j < p; ++j) chi[(size_t)j * N + i] = data[(size_t)j * N + i];   // X_1 = y
      }
      for (int r = 0; r < p; ++r) L[(size_t)tri(r, r) * N + i] = (T)cfg.init_scale_chi;   // S_1 = scale * I
    }
    theta.assign(theta0, theta0 + dt);
    Ltheta.assign(ntri(dt), 0.0);
    if (chol0) std::copy(chol0, chol0 + ntri(dt), Ltheta.begin());
    else for (int r = 0; r < dt; ++r) Ltheta[tri(r, r)] = 0.1;
    t = 0; trace.clear(); mom_count = 0;
    counters.assign((size_t)N, 0u);
    mom_mean.assign((size_t)p * N, 0.0); mom_M2.assign((size_t)p * N, 0.0);
    stats = oracle_stats{};
    have_init = true;
    return ORACLE_OK;
  }

  int get_state(double* c, double* l, double* th, double* lth, int64_t* tt) override {
    if (!have_init) return ORACLE_E_STATE;
    if (c) for (size_t k = 0; k < chi.size(); ++k) c[k] = (double)chi[k];
    if (l) for (size_t k = 0; k < L.size(); ++k) l[k] = (double)L[k];
    if (th) std::copy(theta.begin(), theta.end(), th);
    if (lth) std::copy(Ltheta.begin(), Ltheta.end(), lth);
    if (tt) *tt = t;
    return ORACLE_OK;
  }
  int set_state(const double* c, const double* l, const double* th, const double* lth, int64_t tt) override {
    if (!have_init) return ORACLE_E_STATE;
    if (c) for (size_t k = 0; k < chi.size(); ++k) chi[k] = (T)c[k];
    if (l) for (size_t k = 0; k < L.size(); ++k) L[k] = (T)l[k];
    if (th) std::copy(th, th + dims.dtheta, theta.begin());
    if (lth) std::copy(lth, lth + ntri(dims.dtheta), Ltheta.begin());
    t = tt;
    counters.assign((size_t)cfg.n_objects, (uint32_t)tt);   // as if every object had been updated in every iteration
    return ORACLE_OK;
  }

  // one Gibbs iteration = the plate sweep (O1-O4, moments) followed by the theta decision (O5-O8).  The two halves are
  // separate so that a sharded population can sum its shards' totals in between (oracle_shard_sweep / _decide).
  double zth_[8] = {0}, thp_[8] = {0}, eta_ = 0.0;

  int step(int64_t burn_in, int32_t thin, oracle_taps* taps) override {
    double tot[5];
    int rc = sweep_part(burn_in, taps, tot);
    if (rc != ORACLE_OK) return rc;
    return decide_part(burn_in, thin, taps, tot);
  }

  int sweep_part(int64_t burn_in, oracle_taps* taps, double* tot) override {
    if (!have_init) return ORACLE_E_STATE;
    const int64_t N = cfg.n_objects;
    const int p = dims.p, dt = dims.dtheta, nc = dims.n_cols, nt = ntri(p);
    const int model = cfg.model;

    // O1: this is RAM iteration n = t + 1 (X_1, S_1 are the initial values)
    const uint32_t tcur = (uint32_t)(t + 1);
    const double n_ram = (double)(t + 1) + 1.0;
    double eta = std::pow(n_ram, -cfg.eta_exponent);                // eta_n = n^(-2/3)
    if (cfg.adapt_until > 0 && (t + 1) > cfg.adapt_until) eta = 0.0; // adaptation frozen: S_n = S_{n-1}
    eta_ = eta;

    // O2: theta proposal theta' = theta + L_theta z  (drawn before the sweep: it does not depend on chi)
    double* zth = zth_;
    double* thp = thp_;
    for (int r = 0; r < 8; ++r) { zth[r] = 0.0; thp[r] = 0.0; }
    if (!cfg.freeze_theta) {
      normals_f64(cfg.seed, ORACLE_KIND_THETA, 0, tcur, dt, zth);
      for (int r = 0; r < dt; ++r) {
        double s = theta[r];
        for (int k = 0; k <= r; ++k) s += Ltheta[tri(r, k)] * zth[k];
        thp[r] = s;
      }
    } else {
      for (int r = 0; r < dt; ++r) thp[r] = theta[r];
    }
    T thT[8];
    for (int r = 0; r < dt; ++r) thT[r] = (T)theta[r];
    const T* cT = consts_T.empty() ? nullptr : consts_T.data();
    const double* cD = consts.empty() ? nullptr : consts.data();
    int64_t n_acc = 0, n_nan = 0;

    // O3/O4: plate sweep in index order
    long double S = 0.0L, Delta = 0.0L;
    for (int64_t i = 0; i < N; ++i) {
      T x[8], y[8], z[8] = {}, l[36], d[16], u;
      for (int j = 0; j < p; ++j) x[j] = chi[(size_t)j * N + i];
      for (int k = 0; k < nt; ++k) l[k] = L[(size_t)k * N + i];
      for (int c = 0; c < nc; ++c) d[c] = data[(size_t)c * N + i];
      if (!mask.empty() && !mask[(size_t)i]) {
        // a member held fixed: no RAM step, but it stays in the population sums
        double xd[8], dd[16];
        for (int j = 0; j < p; ++j) xd[j] = (double)x[j];
        for (int c = 0; c < nc; ++c) dd[c] = (double)d[c];
        const double a = logpop<double>(model, xd, dd, theta.data(), cD);
        const double b = logpop<double>(model, xd, dd, thp_, cD);
        S += (long double)a;
        Delta += (long double)(b - a);
        if (taps) {
          const T pc = loglik<T>(model, x, d, cT) + logpop<T>(model, x, d, thT, cT);
          if (taps->chi_prop) for (int j = 0; j < p; ++j) taps->chi_prop[(size_t)j * N + i] = (double)x[j];
          if (taps->pi_cur) taps->pi_cur[i] = (double)pc;
          if (taps->pi_prop) taps->pi_prop[i] = (double)pc;
          if (taps->alpha) taps->alpha[i] = 0.0;
          if (taps->u) taps->u[i] = 1.0;
          if (taps->accepted) taps->accepted[i] = 0;
          if (taps->L_new) for (int k = 0; k < nt; ++k) taps->L_new[(size_t)k * N + i] = (double)l[k];
          if (taps->a) taps->a[i] = a;
          if (taps->b) taps->b[i] = b;
        }
        if (cfg.keep_chi_moments && (t + 1) > burn_in) {
          const double k1 = (double)(mom_count + 1);
          for (int j = 0; j < p; ++j) {
            const size_t q = (size_t)j * N + i;
            const double dl = xd[j] - mom_mean[q];
            mom_mean[q] += dl / k1;
            mom_M2[q] += dl * (xd[j] - mom_mean[q]);
          }
        }
        continue;
      }
      // eta_n of THIS object: its own update count when asked for (n_i = count + 2: the first update is n = 2)
      double eta_i = eta;
      if (cfg.per_object_counter && eta != 0.0) eta_i = std::pow((double)counters[(size_t)i] + 2.0, -cfg.eta_exponent);
      counters[(size_t)i] += 1u;
      if (sizeof(T) == 8) {
        double zz[8] = {}, uu = 0;
        plate_draws_f64(cfg.seed, (uint64_t)(cfg.object_offset + i), tcur, p, zz, &uu);
        for (int j = 0; j < p; ++j) z[j] = (T)zz[j];
        u = (T)uu;
      } else {
        float zf[2] = {0.0f, 0.0f}, uf;
        plate_draws_f32(cfg.seed, (uint64_t)(cfg.object_offset + i), tcur, p, zf, &uf);
        z[0] = (T)zf[0]; z[1] = (T)zf[1]; u = (T)uf;
        if (p == 1) z[1] = T(0);
      }
      // step 1: Y = X + S U
      for (int r = 0; r < p; ++r) {
        T s = x[r];
        for (int k = 0; k <= r; ++k) s += l[tri(r, k)] * z[k];
        y[r] = s;
      }
      // step 2: alpha = min{1, pi(Y)/pi(X)}, pi = l_i * f(.;theta)
      const T pc = loglik<T>(model, x, d, cT) + logpop<T>(model, x, d, thT, cT);
      const T pp = loglik<T>(model, y, d, cT) + logpop<T>(model, y, d, thT, cT);
      const T diff = pp - pc;
      T la;
      if (std::isnan(diff)) { la = -std::numeric_limits<T>::infinity(); n_nan++; }
      else la = std::min(T(0), diff);
      const T alpha = std::exp(la);
      const bool acc = (u < alpha);
      if (acc) { for (int j = 0; j < p; ++j) x[j] = y[j]; n_acc++; }
      // step 3: S_n = chol(S (I + eta (alpha - alpha_*) U U^T/||U||^2) S^T)
      T lnew[36];
      ram_update<T>(p, l, z, (T)eta_i * (alpha - (T)cfg.target_accept_chi), lnew);
      for (int j = 0; j < p; ++j) chi[(size_t)j * N + i] = x[j];
      for (int k = 0; k < nt; ++k) L[(size_t)k * N + i] = lnew[k];
      // population terms at the new chi, fp64 (log-posterior with the updated parameters)
      double xd[8], dd[16];
      for (int j = 0; j < p; ++j) xd[j] = (double)x[j];
      for (int c = 0; c < nc; ++c) dd[c] = (double)d[c];
      const double a = logpop<double>(model, xd, dd, theta.data(), cD);
      const double b = logpop<double>(model, xd, dd, thp_, cD);
      S += (long double)a;
      Delta += (long double)(b - a);
      if (taps) {
        if (taps->chi_prop) for (int j = 0; j < p; ++j) taps->chi_prop[(size_t)j * N + i] = (double)y[j];
        if (taps->pi_cur) taps->pi_cur[i] = (double)pc;
        if (taps->pi_prop) taps->pi_prop[i] = (double)pp;
        if (taps->alpha) taps->alpha[i] = (double)alpha;
        if (taps->u) taps->u[i] = (double)u;
        if (taps->accepted) taps->accepted[i] = acc ? 1 : 0;
        if (taps->L_new) for (int k = 0; k < nt; ++k) taps->L_new[(size_t)k * N + i] = (double)lnew[k];
        if (taps->a) taps->a[i] = a;
        if (taps->b) taps->b[i] = b;
      }
      // O8 (plate part): running moments after burn-in (Welford)
      if (cfg.keep_chi_moments && (t + 1) > burn_in) {
        const double k1 = (double)(mom_count + 1);
        for (int j = 0; j < p; ++j) {
          const size_t q = (size_t)j * N + i;
          const double dl = xd[j] - mom_mean[q];
          mom_mean[q] += dl / k1;
          mom_M2[q] += dl * (xd[j] - mom_mean[q]);
        }
      }
    }
    if (cfg.keep_chi_moments && (t + 1) > burn_in) { mom_count++; stats.moment_samples = mom_count; }
    tot[0] = (double)S; tot[1] = (double)Delta; tot[2] = 0.0; tot[3] = (double)n_acc; tot[4] = (double)n_nan;
    return ORACLE_OK;
  }

  // tot = {S, Delta, -, n_accept, n_nonfinite} summed over the whole population (all shards)
  int decide_part(int64_t burn_in, int32_t thin, oracle_taps* taps, const double* tot) override {
    if (!have_init) return ORACLE_E_STATE;
    const int dt = dims.dtheta;
    const int model = cfg.model;
    const double ninf = -std::numeric_limits<double>::infinity();
    const uint32_t tcur = (uint32_t)(t + 1);
    const double eta = eta_;
    const double* zth = zth_;
    const double* thp = thp_;
    const double S = tot[0], Delta = tot[1];
    stats.chi_accepts += (int64_t)tot[3];
    stats.nonfinite += (int64_t)tot[4];
    stats.chi_proposals += mask.empty() ? (cfg.n_objects_total ? cfg.n_objects_total : cfg.n_objects) : n_active();

    // O5-O7: theta decision and RAM update of L_theta
    double T_cur = 0, T_prop = 0, lp_cur = 0, lp_prop = 0, log_r = 0, alpha_th = 0, u_th = 0;
    int acc_th = 0;
    if (!cfg.freeze_theta) {
      T_cur = theta_only(theta.data());
      lp_cur = logprior(model, theta.data()) + user_prior(theta.data());
      lp_prop = logprior(model, thp) + user_prior(thp);
      double la_th;
      // Eq. 4.3 divides by I(theta')^N: where the selection integral is not a positive normal number the likelihood is
      // undefined and the proposal is rejected like one outside the prior's support (reading R26)
      bool undefined = false;
      if (model == M_BB1_FLUXNOISE1D && lp_prop != ninf)
        undefined = !(table.bb1_integral(thp, consts.data()) >= std::numeric_limits<double>::min());
      if (lp_prop == ninf || undefined) { log_r = ninf; la_th = ninf; T_prop = 0; }
      else {
        T_prop = theta_only(thp);
        log_r = (double)Delta + (T_prop - T_cur) + (lp_prop - lp_cur);
        la_th = std::isnan(log_r) ? ninf : std::min(0.0, log_r);
      }
      alpha_th = std::exp(la_th);
      u_th = accept_uniform_f64(cfg.seed, ORACLE_KIND_THETA, 0, tcur);
      acc_th = (u_th < alpha_th) ? 1 : 0;
      if (acc_th) { for (int r = 0; r < dt; ++r) theta[r] = thp[r]; stats.theta_accepts++; }
      stats.theta_proposals++;
      std::vector<double> lnew(ntri(dt));
      ram_update<double>(dt, Ltheta.data(), zth, eta * (alpha_th - cfg.target_accept_theta), lnew.data());
      Ltheta = lnew;
    }
    if (taps) {
      for (int r = 0; r < 8; ++r) taps->theta_prop[r] = r < dt ? thp[r] : 0.0;
      taps->S = (double)S; taps->Delta = (double)Delta; taps->T_cur = T_cur; taps->T_prop = T_prop;
      taps->lp_cur = lp_cur; taps->lp_prop = lp_prop; taps->log_r = log_r; taps->alpha_theta = alpha_th;
      taps->u_theta = u_th; taps->accepted_theta = acc_th;
    }
    t += 1;
    stats.iterations = t;
    // O8 (theta part): thinned trace
    if (t > burn_in && thin > 0 && ((t - burn_in) % thin) == 0) {
      trace.insert(trace.end(), theta.begin(), theta.end());
      stats.trace_rows = (int64_t)(trace.size() / dt);
    }
    return ORACLE_OK;
  }
};

}  // namespace oracle

struct oracle_sampler { std::unique_ptr<oracle::Base> impl; };

using namespace oracle;

extern "C" {

int oracle_model_dims(int model, int* p, int* dtheta, int* n_data_cols, int* n_consts) {
  Dims d;
  if (!model_dims(model, &d)) return ORACLE_E_INVALID;
  if (p) *p = d.p;
  if (dtheta) *dtheta = d.dtheta;
  if (n_data_cols) *n_data_cols = d.n_cols;
  if (n_consts) *n_consts = d.n_consts;
  return ORACLE_OK;
}

int oracle_create(const oracle_config* cfg, oracle_sampler** out) {
  if (!cfg || !out) return ORACLE_E_INVALID;
  Dims d;
  if (!model_dims(cfg->model, &d) || cfg->n_objects < 0) return ORACLE_E_INVALID;
  if (!(cfg->target_accept_chi > 0 && cfg->target_accept_chi < 1)) return ORACLE_E_INVALID;
  if (!(cfg->target_accept_theta > 0 && cfg->target_accept_theta < 1)) return ORACLE_E_INVALID;
  if (cfg->object_offset < 0 || (cfg->object_offset & 1) || cfg->n_objects_total < 0) return ORACLE_E_INVALID;
  std::unique_ptr<Base> b;
  if (cfg->precision == ORACLE_F64) b.reset(new Impl<double>());
  else if (cfg->precision == ORACLE_F32_STATE_F64_REDUCE && d.p <= 2) b.reset(new Impl<float>());   // fp32 draws: p <= 2
  else return ORACLE_E_UNSUPPORTED;
  b->cfg = *cfg;
  b->dims = d;
  *out = new oracle_sampler{std::move(b)};
  return ORACLE_OK;
}

void oracle_destroy(oracle_sampler* s) { delete s; }

int oracle_set_data(oracle_sampler* s, const double* const* cols, int n_cols) {
  if (!s || !cols) return ORACLE_E_INVALID;
  return s->impl->set_data(cols, n_cols);
}

int oracle_set_model_consts(oracle_sampler* s, const double* v, int n) {
  if (!s) return ORACLE_E_INVALID;
  Base* b = s->impl.get();
  if (n != b->dims.n_consts) return ORACLE_E_INVALID;
  b->consts.assign(v, v + n);
  if (b->cfg.precision == ORACLE_F32_STATE_F64_REDUCE) {
    auto* f = static_cast<Impl<float>*>(b);
    f->consts_T.resize(n);
    for (int k = 0; k < n; ++k) f->consts_T[k] = (float)v[k];
  } else {
    auto* f = static_cast<Impl<double>*>(b);
    f->consts_T.assign(v, v + n);
  }
  if (b->cfg.model == M_THINNED_SCHECHTER1D) b->table.build(b->consts.data());
  if (b->cfg.model == M_BB1_FLUXNOISE1D) b->table.build_bb1(b->consts.data());
  b->have_consts = true;
  return ORACLE_OK;
}

int oracle_set_update_mask(oracle_sampler* s, const uint8_t* mask) {
  if (!s) return ORACLE_E_INVALID;
  Base* b = s->impl.get();
  if (mask && b->cfg.n_objects_total != 0 && b->cfg.n_objects_total != b->cfg.n_objects) return ORACLE_E_UNSUPPORTED;
  if (mask) b->mask.assign(mask, mask + b->cfg.n_objects);
  else b->mask.clear();
  return ORACLE_OK;
}
int oracle_get_counters(oracle_sampler* s, uint32_t* out) {
  if (!s || !out) return ORACLE_E_INVALID;
  if (!s->impl->have_init) return ORACLE_E_STATE;
  std::copy(s->impl->counters.begin(), s->impl->counters.end(), out);
  return ORACLE_OK;
}
int oracle_set_counters(oracle_sampler* s, const uint32_t* in) {
  if (!s || !in) return ORACLE_E_INVALID;
  if (!s->impl->have_init) return ORACLE_E_STATE;
  s->impl->counters.assign(in, in + s->impl->cfg.n_objects);
  return ORACLE_OK;
}

int oracle_set_init(oracle_sampler* s, const double* chi0, const double* theta0, const double* chol0) {
  if (!s || !theta0) return ORACLE_E_INVALID;
  return s->impl->set_init(chi0, theta0, chol0);
}

int oracle_step(oracle_sampler* s, int64_t burn_in, int32_t thin, oracle_taps* taps) {
  if (!s || thin < 1 || burn_in < 0) return ORACLE_E_INVALID;
  return s->impl->step(burn_in, thin, taps);
}

int oracle_shard_sweep(oracle_sampler* s, int64_t burn_in, int32_t thin, double* totals) {
  if (!s || !totals || thin < 1 || burn_in < 0) return ORACLE_E_INVALID;
  return s->impl->sweep_part(burn_in, nullptr, totals);
}
int oracle_shard_decide(oracle_sampler* s, int64_t burn_in, int32_t thin, const double* totals_global) {
  if (!s || !totals_global || thin < 1 || burn_in < 0) return ORACLE_E_INVALID;
  return s->impl->decide_part(burn_in, thin, nullptr, totals_global);
}

int oracle_run(oracle_sampler* s, int64_t n_iter, int64_t burn_in, int32_t thin) {
  if (!s || n_iter < 0 || thin < 1 || burn_in < 0) return ORACLE_E_INVALID;
  for (int64_t k = 0; k < n_iter; ++k) {
    const int rc = s->impl->step(burn_in, thin, nullptr);
    if (rc != ORACLE_OK) return rc;
  }
  return ORACLE_OK;
}

int oracle_get_theta_trace(oracle_sampler* s, double* out, int64_t cap_rows, int64_t* n_rows) {
  if (!s || !n_rows) return ORACLE_E_INVALID;
  Base* b = s->impl.get();
  const int64_t rows = (int64_t)(b->trace.size() / b->dims.dtheta);
  *n_rows = rows;
  if (!out) return ORACLE_OK;
  if (cap_rows < rows) return ORACLE_E_INVALID;
  std::copy(b->trace.begin(), b->trace.end(), out);
  return ORACLE_OK;
}

int oracle_get_chi_moments(oracle_sampler* s, double* mean, double* var, int64_t cap_objects, int64_t* n_samples) {
  if (!s || !n_samples) return ORACLE_E_INVALID;
  Base* b = s->impl.get();
  if (!b->cfg.keep_chi_moments) return ORACLE_E_STATE;
  *n_samples = b->mom_count;
  if (cap_objects < b->cfg.n_objects) return ORACLE_E_INVALID;
  const size_t n = b->mom_mean.size();
  for (size_t k = 0; k < n; ++k) {
    if (mean) mean[k] = b->mom_mean[k];
    if (var) var[k] = b->mom_count > 1 ? b->mom_M2[k] / (double)(b->mom_count - 1) : 0.0;
  }
  return ORACLE_OK;
}

int oracle_get_state(oracle_sampler* s, double* chi, double* L, double* theta, double* L_theta, int64_t* t) {
  if (!s) return ORACLE_E_INVALID;
  return s->impl->get_state(chi, L, theta, L_theta, t);
}
int oracle_set_state(oracle_sampler* s, const double* chi, const double* L, const double* theta,
                     const double* L_theta, int64_t t) {
  if (!s || t < 0) return ORACLE_E_INVALID;
  return s->impl->set_state(chi, L, theta, L_theta, t);
}

int oracle_get_stats(oracle_sampler* s, oracle_stats* out) {
  if (!s || !out) return ORACLE_E_INVALID;
  *out = s->impl->stats;
  return ORACLE_OK;
}

int oracle_theta_only(oracle_sampler* s, const double* theta, double* out) {
  if (!s || !theta || !out) return ORACLE_E_INVALID;
  if (s->impl->dims.n_consts > 0 && !s->impl->have_consts) return ORACLE_E_STATE;
  *out = s->impl->theta_only(theta);
  return ORACLE_OK;
}

int oracle_get_selection_table(oracle_sampler* s, double* xk, double* Wk, int cap, int* n) {
  if (!s || !n) return ORACLE_E_INVALID;
  Base* b = s->impl.get();
  *n = (int)b->table.xk.size();
  if (cap < *n) return ORACLE_E_INVALID;
  std::copy(b->table.xk.begin(), b->table.xk.end(), xk);
  std::copy(b->table.Wk.begin(), b->table.Wk.end(), Wk);
  return ORACLE_OK;
}

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const Words r = philox4x32_10(ctr, key);
  for (int k = 0; k < 4; ++k) out[k] = r.w[k];
}
void oracle_stream_words(uint64_t seed, int kind, uint64_t obj, uint32_t t, uint32_t d, uint32_t out[4]) {
  const Words r = stream_words(seed, kind, obj, t, d);
  for (int k = 0; k < 4; ++k) out[k] = r.w[k];
}
double oracle_uniform_f64(uint64_t seed, int kind, uint64_t obj, uint32_t t, uint32_t d) {
  const Words r = stream_words(seed, kind, obj, t, d);
  return u01_f64(r.w[0], r.w[1]);
}
void oracle_normals_f64(uint64_t seed, int kind, uint64_t obj, uint32_t t, int n, double* z) {
  normals_f64(seed, kind, obj, t, n, z);
}
void oracle_draws_f32(uint64_t seed, int kind, uint64_t obj, uint32_t t, float* z2, float* u) {
  draws_f32(seed, kind, obj, t, z2, u);
}
void oracle_plate_draws_f64(uint64_t seed, uint64_t i, uint32_t t, int p, double* z, double* u) {
  plate_draws_f64(seed, i, t, p, z, u);
}
void oracle_plate_draws_f32(uint64_t seed, uint64_t i, uint32_t t, int p, float* z, float* u) {
  plate_draws_f32(seed, i, t, p, z, u);
}
double oracle_loglik(int model, const double* chi, const double* d, const double* consts) {
  return loglik<double>(model, chi, d, consts);
}
double oracle_logpop(int model, const double* chi, const double* d, const double* th, const double* consts) {
  return logpop<double>(model, chi, d, th, consts);
}
float oracle_loglik_f32(int model, const float* chi, const float* d, const float* consts) {
  return loglik<float>(model, chi, d, consts);
}
float oracle_logpop_f32(int model, const float* chi, const float* d, const float* th, const float* consts) {
  return logpop<float>(model, chi, d, th, consts);
}
double oracle_logprior(int model, const double* theta) { return logprior(model, theta); }
void oracle_ram_update(int p, const double* L_packed, const double* z, double c, double* L_out) {
  if (p < 1 || p > 8) return;
  ram_update<double>(p, L_packed, z, c, L_out);
}
void oracle_gauss_legendre(int n, double a, double b, double* x, double* w) { gauss_legendre(n, a, b, x, w); }
double oracle_bb1_log_norm(double beta, double l, double u) { return bb1_log_norm(beta, l, u); }
double oracle_bb1_selection_integral_2d(const double* theta, const double* consts) {
  return SelectionTable::selection_integral_2d(theta, consts);
}
double oracle_sum(const double* v, int64_t n) {
  long double acc = 0.0L;
  for (int64_t i = 0; i < n; ++i) acc += (long double)v[i];
  return (double)acc;
}

}  // extern "C"
