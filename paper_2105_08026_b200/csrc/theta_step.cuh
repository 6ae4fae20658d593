// theta_step.cuh -- the theta Metropolis-Hastings tail (PAPER.md:108 Eq. 2.5, :142), host + device.
//
// Two implementations of the same arithmetic:
//   (a) serial, __host__ __device__: `prepare_iteration` + `tail_decide`.  Used on the host (THETA_HOST, the
//       paper's own split) and once per set_init / set_state on the device (k_init_iter).
//   (b) block-parallel, device only: `tail_block`.  Used by the persistent kernel (every block, redundantly and
//       bit-identically) and by k_tail (THETA_GRAPH, debug_step).  The serial chain of (a) costs ~4.4 us per
//       iteration on one thread (profiles/r01a); (b) takes everything that does not depend on the decision off
//       the critical path (draws are made two iterations ahead while warp 0 waits for the other blocks'
//       partials) and spreads the rest over lanes and warps.
#pragma once
#include "models.cuh"

namespace hm {

constexpr int MAXD = 8;                       // max dtheta
constexpr int MAXTRI = MAXD * (MAXD + 1) / 2;
constexpr int NPART = 5;                      // per-block partials: S, Delta, Tq, n_accept, n_nonfinite

// Decision-independent quantities of one iteration t; ring slot t % 3 of Iter::dr.
struct Draws {
  double z[MAXD];       // z_theta ~ N(0, I)                       (theta Philox stream, draws 1..)
  double uh[MAXD];      // z / |z|
  double Pc[MAXD + 1];  // Pc[j] = sum_{k<j} uh_k^2
  double eta;           // eta_n = n^(-eta_exp), n = t + 1         (X_1, S_1 are initial values)
  double u;             // accept uniform of the theta step        (theta Philox stream, draw 0)
  double lu;            // ln u (device tail: the decision is taken as ln u < ln alpha, see decide_scalars)
};

// Iteration state: lives in global memory between launches, in shared memory inside the kernels.
struct Iter {
  double theta[MAXD], thetaP[MAXD];   // theta and the pre-drawn proposal theta' of the PREPARED iteration t
  double Lth[MAXTRI];                 // packed lower-triangular proposal factor of the theta RAM
  double W[MAXTRI];                   // W[tri(i,j)] = sum_{k=j+1..i} Lth[i,k] uh_k for iteration t
  Draws dr[3];                        // slots t%3 (iteration t) and (t+1)%3 are valid; (t+2)%3 is scratch
  ThetaK kc, kp;                      // theta-derived constants at theta / theta'
  double T_cur, lp_cur, lp_prop;      // theta-only term and log prior at theta; log prior at theta'
  double lp_prop_next;                // staging slot of the block-parallel tail
  double inv_k;                       // 1 / (mom_count + 1) of the PREPARED iteration (Welford step of the running chi moments)
  // taps of the last decision (debug_step / host mode read them)
  double S, Delta, T_prop, log_r, alpha_theta, u_theta, T_cur_used, lp_cur_used, tap_thetaP[MAXD];
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
  double n_objects;     // N of the selection term -N log I(theta) (M4)
  long long adapt_until;             // 0: adapt forever; else eta_n = 0 for t > adapt_until
  double prior_mean[MAXD], prior_isd[MAXD];   // user prior: independent normal factors on theta (isd = 0: none)
};

// eta_n of iteration t (n = t + 1: X_1, S_1 are the initial values); 0 once adaptation is frozen
HM_HD double eta_of(const TailCfg& c, long long t) {
  if (c.adapt_until > 0 && t > c.adapt_until) return 0.0;
  return pow((double)(t + 1), -c.eta_exp);
}
// log prior = the model's default (uniform on a box; models.cuh) + the user's normal factors
HM_HD double log_prior_full(const TailCfg& c, const double* th, int model) {
  double s = log_prior(model, th);
  for (int j = 0; j < c.dtheta; ++j) {
    const double r = (th[j] - c.prior_mean[j]) * c.prior_isd[j];
    s += -0.5 * r * r;
  }
  return s;
}
HM_HD double log_prior_full(const TailCfg& c, const double* th) { return log_prior_full(c, th, c.model); }

// ring slot of iteration t (t < 2^32 is checked by cudahm_run): a 32-bit modulo by a constant, not the 64-bit software routine
HM_HD int slot3(long long t) { return (int)((unsigned)t % 3u); }

HM_HD int tri(int r, int c) { return r * (r + 1) / 2 + c; }
HM_HD int tri_row(int e) { int r = 0; while ((r + 1) * (r + 2) / 2 <= e) ++r; return r; }

// ---------------------------------------------------------------------------------------------------
// RAM step 3 (Eq. 2.6) for general p as a rank-one update in closed form:
//   chol(I + c u u^T) = K,  K_jj = sqrt(s_{j+1}/s_j),  K_ij = c u_i u_j / sqrt(s_j s_{j+1}) (i > j),
//   s_j = 1 + c sum_{k<j} u_k^2;  then L <- L K, lower-triangular with positive diagonal, and
//   (L K)(L K)^T = L (I + c u u^T) L^T, hence THE left Cholesky factor.
//   1 + c >= 1 - alpha_* > 0, so every s_j > 0.  Entry-wise:
//   (L K)_ij = L_ij Kd_j + g_j W_ij,  Kd_j = rs_{j+1}/rs_j,  g_j = c u_j/(rs_j rs_{j+1}),  rs_j = sqrt(s_j),
//   W_ij = sum_{k=j+1..i} L_ik u_k (does not depend on c: precomputed off the critical path).
HM_HD void ram_coeffs(int j, double c, const Draws& d, double* Kd, double* g) {
  const double s0 = 1.0 + c * d.Pc[j], s1 = 1.0 + c * d.Pc[j + 1];
#ifdef __CUDA_ARCH__
  const double r = rsqrt(s0 * s1);          // one reciprocal square root instead of two roots and two divisions
#else
  const double r = 1.0 / sqrt(s0 * s1);
#endif
  *Kd = s1 * r;                             // sqrt(s1/s0)
  *g = c * d.uh[j] * r;                     // c u_j / sqrt(s0 s1)
}

HM_HD void make_draws(Draws& d, const TailCfg& c, long long t) {
  d.eta = eta_of(c, t);
  for (int j = 0; j < MAXD; ++j) { d.z[j] = 0.0; d.uh[j] = 0.0; }
  for (int j = 0; j <= MAXD; ++j) d.Pc[j] = 0.0;
  d.u = 0.0; d.lu = 0.0;
  if (c.freeze_theta) return;
  normals(c.seed, KIND_THETA, 0ull, (uint32_t)t, c.dtheta, d.z);
  double n2 = 0.0;
  for (int j = 0; j < c.dtheta; ++j) n2 += d.z[j] * d.z[j];
  const double rn = 1.0 / sqrt(n2);
  double s = 0.0;
  for (int j = 0; j < c.dtheta; ++j) { d.uh[j] = d.z[j] * rn; d.Pc[j] = s; s += d.uh[j] * d.uh[j]; }
  d.Pc[c.dtheta] = s;
  const U4 r = stream(c.seed, KIND_THETA, 0ull, (uint32_t)t, 0u);
  d.u = u01(r.x, r.y);
  d.lu = hm_log_any_pos(d.u);
}

HM_HD double make_W_entry(const Iter& it, const Draws& d, int i, int j) {
  double w = 0.0;
  for (int k = i; k > j; --k) w += it.Lth[tri(i, k)] * d.uh[k];
  return w;
}

HM_HD double propose_entry(const Iter& it, const Draws& d, int r) {
  double s = it.theta[r];
  for (int k = 0; k <= r; ++k) s += it.Lth[tri(r, k)] * d.z[k];
  return s;
}

// (a) serial: everything about iteration t that does not depend on its sweep.  theta' = theta + L_theta z is
// drawn BEFORE the sweep so one pass evaluates f at theta and theta' (reading R7).
HM_HD void prepare_iteration(Iter& it, const TailCfg& c, long long t) {
  it.t = t;
  Draws& d = it.dr[slot3(t)];
  make_draws(d, c, t);
  make_draws(it.dr[slot3(t + 1)], c, t + 1);
  it.inv_k = 1.0 / (double)(it.mom_count + 1);
  if (!c.freeze_theta) {
    for (int r = 0; r < c.dtheta; ++r) it.thetaP[r] = propose_entry(it, d, r);
    for (int i = 0; i < c.dtheta; ++i)
      for (int j = 0; j <= i; ++j) it.W[tri(i, j)] = make_W_entry(it, d, i, j);
    it.kp = theta_consts(c.model, it.thetaP);
    it.lp_prop = log_prior_full(c, it.thetaP);
  } else {
    for (int r = 0; r < c.dtheta; ++r) it.thetaP[r] = it.theta[r];
    it.kp = it.kc;
    it.lp_prop = it.lp_cur;
  }
}

// The acceptance part shared by (a) and (b): log r, ln alpha = min(0, log r), accept flag.
// The paper's rule is "accept iff u < alpha"; it is taken here as ln u < ln alpha with ln u drawn
// ahead of time, so that no exponential sits between the arrival of the sums and the decision the next sweep is
// waiting for.  The two forms differ only where |ln alpha - ln u| is of the order of one rounding error, far
// inside the near-tie band (1e-9) in which BASELINE.json allows accept sequences to differ.  alpha itself (the
// RAM update needs it) is computed by the caller afterwards.
HM_HD void decide_scalars(const Iter& it, const TailCfg& c, const Draws& d, double Delta, double tq, double* T_prop,
                          double* log_r, double* la, int* acc, int model = -1) {
  if (model < 0) model = c.model;
  *T_prop = 0.0;
  // M4: Eq. 4.3 divides by I(theta')^N; a selection sum that is not a positive normal number leaves the likelihood undefined
  // and the proposal is rejected like one outside the prior's support (reading R26; hm_log_pos needs a normal input)
  const bool undefined = model == M_BB1_FLUXNOISE1D && !(tq >= 2.2250738585072014e-308);
  if (it.lp_prop == -INFINITY || undefined) {
    *log_r = -INFINITY; *la = -INFINITY;
  } else {
    // M1: T(theta') = -A' sum_k W_k phi(x_k; theta'): minus the expected detected count (Eq. 4.4 denominator)
    // M4: T(theta') = -N log sum_k W_k rho(x_k; theta')   (Eq. 4.3-4.4)
    *T_prop = theta_only_from_sum(model, it.kp, tq, c.n_objects);
    *log_r = Delta + (*T_prop - it.T_cur) + (it.lp_prop - it.lp_cur);
    *la = (*log_r != *log_r) ? -INFINITY : fmin(0.0, *log_r);
  }
  *acc = d.lu < *la ? 1 : 0;
}

// bookkeeping shared by (a) and (b): taps and counters fed by the sweep totals ...
HM_HD void decide_counters(Iter& it, double S, double Delta, double nacc, double nnan) {
  it.S = S;
  it.Delta = Delta;
  it.chi_acc += (unsigned long long)nacc;
  it.nonfinite += (unsigned long long)nnan;
}
// ... and the moments count / trace row of iteration it.t (independent of the decision)
HM_HD void decide_schedule(Iter& it, const TailCfg& c) {
  if (c.keep_moments && it.t > c.burn_in) it.mom_count += 1;
  it.inv_k = 1.0 / (double)(it.mom_count + 1);      // for the sweep of iteration t + 1: one division here instead of one per thread
  it.trace_write = 0;
  if (it.t > c.burn_in && ((it.t - c.burn_in) % c.thin) == 0 && it.trace_rows < c.max_trace_rows) {
    it.trace_rows += 1;
    it.trace_write = 1;
  }
}

// (a) serial: the theta decision of iteration it.t from the reduced sweep totals {S, Delta, Tq, nacc, nnan}.
// Sets it.trace_write when the (new) theta has to be appended to the thinned trace at row it.trace_rows - 1.
HM_HD void tail_decide(Iter& it, const TailCfg& c, const double* tot) {
  const Draws& d = it.dr[slot3(it.t)];
  it.accepted_theta = 0;
  it.T_prop = 0.0; it.log_r = 0.0; it.alpha_theta = 0.0; it.u_theta = 0.0;
  it.T_cur_used = it.T_cur; it.lp_cur_used = it.lp_cur;
  for (int r = 0; r < MAXD; ++r) it.tap_thetaP[r] = it.thetaP[r];
  if (!c.freeze_theta) {
    int acc;
    double la;
    decide_scalars(it, c, d, tot[1], tot[2], &it.T_prop, &it.log_r, &la, &acc);
    it.alpha_theta = hm_exp_any(la);
    it.u_theta = d.u;
    it.theta_prop_n += 1;
    if (acc) {
      it.accepted_theta = 1;
      it.theta_acc += 1;
      for (int r = 0; r < c.dtheta; ++r) it.theta[r] = it.thetaP[r];
      it.kc = it.kp; it.T_cur = it.T_prop; it.lp_cur = it.lp_prop;
    }
    const double cc = d.eta * (it.alpha_theta - c.astar_theta);
    for (int j = 0; j < c.dtheta; ++j) {
      double Kd, g;
      ram_coeffs(j, cc, d, &Kd, &g);
      for (int i = j; i < c.dtheta; ++i) it.Lth[tri(i, j)] = it.Lth[tri(i, j)] * Kd + g * it.W[tri(i, j)];
    }
  }
  decide_counters(it, tot[0], tot[1], tot[3], tot[4]);
  decide_schedule(it, c);
}

#ifdef __CUDACC__
// ---------------------------------------------------------------------------------------------------
// (b) block-parallel tail (device).  Called by 4 warps (`warp` = 0..3 among them; `sync` = a barrier over exactly
// those 128 threads); `it` is in shared memory.  tot = {S, Delta, Tq, nacc, nnan}, valid in every lane of warp 0
// (S, nacc, nnan feed only the tap and the counters: the persistent kernels pass zeros and count locally).
// Decides iteration t = it.t, prepares iteration t + 1 and makes the draws of iteration t + 2.
//
//   phase B   warp 0:  decision scalars (all lanes redundantly) -> RAM coefficients (lane j) -> new L_theta
//                      (lane e) -> theta, theta' of t+1 (lane r) -> kc <- kp on accept (lane v).
//             warp 1:  z, uh, Pc of iteration t+2 (Box-Muller pair per lane);  warp 2: eta of t+2, moments /
//             trace schedule of t;  warp 3: accept uniform of t+2.  None of these depends on the decision, so
//             they run while warp 0 is still waiting for the other blocks' partials.
//   phase C   warp 0..2: the parts of theta_consts(theta'); warp 3: log prior(theta'); warp 1 also W of t+1
//             (lane e); warp 2 also the trace row.
struct SyncAll { __device__ __forceinline__ void operator()() const { __syncthreads(); } };
template <int ID, int THREADS>
struct SyncNamed {
  __device__ __forceinline__ void operator()() const { asm volatile("bar.sync %0, %1;" ::"n"(ID), "n"(THREADS) : "memory"); }
};

struct NoSignal { __device__ __forceinline__ void operator()() const {} };
template <int ID, int THREADS>
struct ArriveNamed {
  __device__ __forceinline__ void operator()() const {
    // (no fence needed: when the barrier completes, bar.arrive has ordered this thread's prior shared-memory writes for its participants)
    asm volatile("bar.arrive %0, %1;" ::"n"(ID), "n"(THREADS) : "memory");
  }
};

// `decided` is called once by every thread of the four warps as soon as what the next sweep's targets need is
// final: kc (theta_{t+1}'s constants: the accept decision only, NOT the RAM update of L_theta), the moments count
// and eta of iteration t + 1.  theta', kp, the prior, L_theta and W are final only when tail_block returns.
// MODEL: the compiled-in model of the calling kernel (the persistent kernels know it at compile time, which collapses the
// model switches of the tail -- the serial chain every iteration waits for); -1: taken from c.model at run time (k_tail).
template <int MODEL = -1, class Sync, class Decided = NoSignal>
__device__ __forceinline__ void tail_block(Iter& it, const TailCfg& c, const double* tot, double* trace_or_null,
                                           const int warp, const Sync sync, const Decided decided = Decided()) {
  const int lane = threadIdx.x & 31;
  const int model = MODEL >= 0 ? MODEL : c.model;
  const int dt = c.dtheta, nt = dt * (dt + 1) / 2;
  const long long t = it.t;
  const int r0 = slot3(t), r1 = r0 == 2 ? 0 : r0 + 1, r2 = r1 == 2 ? 0 : r1 + 1;
  const Draws& d0 = it.dr[r0];
  const Draws& d1 = it.dr[r1];
  Draws& d2 = it.dr[r2];

  // decision scalars stay in warp 0's registers until phase C, where the taps are written (off the critical path)
  double T_prop = 0.0, log_r = 0.0, alpha = 0.0;
  int acc = 0;
  if (warp == 0) {
    if (!c.freeze_theta) {
      double la;
      decide_scalars(it, c, d0, tot[1], tot[2], &T_prop, &log_r, &la, &acc, model);
      const double kpv = lane < 8 ? it.kp.v[lane] : 0.0;
      if (lane < 8 && acc) it.kc.v[lane] = kpv;          // theta_{t+1}'s constants: all the next sweep's targets need
      decided();
      alpha = hm_exp_any(la);
      const double cc = d0.eta * (alpha - c.astar_theta);
      double Kd = 1.0, g = 0.0;
      if (lane < dt) ram_coeffs(lane, cc, d0, &Kd, &g);
      const int e = lane < nt ? lane : 0;
      const int ei = tri_row(e), ej = e - ei * (ei + 1) / 2;
      const double Kd_j = __shfl_sync(0xffffffffu, Kd, ej), g_j = __shfl_sync(0xffffffffu, g, ej);
      const double l_new = it.Lth[e] * Kd_j + g_j * it.W[e];
      const double th_old = lane < dt ? it.theta[lane] : 0.0, thp_old = lane < dt ? it.thetaP[lane] : 0.0;
      __syncwarp();
      if (lane < nt) it.Lth[e] = l_new;
      if (lane < MAXD) it.tap_thetaP[lane] = lane < dt ? thp_old : 0.0;
      if (lane < dt) it.theta[lane] = acc ? thp_old : th_old;
      __syncwarp();
      if (lane < dt) it.thetaP[lane] = propose_entry(it, d1, lane);
    } else {
      decided();
    }
  } else if (warp == 1) {
    decided();
    if (!c.freeze_theta) {
      if (2 * lane < dt) {
        double rad, cs, sn;
        box_muller(stream(c.seed, KIND_THETA, 0ull, (uint32_t)(t + 2), 1u + (uint32_t)lane), &rad, &cs, &sn);
        d2.z[2 * lane] = rad * cs;
        if (2 * lane + 1 < dt) d2.z[2 * lane + 1] = rad * sn;
      }
      __syncwarp();
      if (lane == 0) {
        double n2 = 0.0;
        for (int j = 0; j < dt; ++j) n2 += d2.z[j] * d2.z[j];
        const double rn = 1.0 / sqrt(n2);
        double s = 0.0;
        for (int j = 0; j < dt; ++j) { d2.uh[j] = d2.z[j] * rn; d2.Pc[j] = s; s += d2.uh[j] * d2.uh[j]; }
        d2.Pc[dt] = s;
      }
    }
  } else if (warp == 2) {
    if (lane == 0) decide_schedule(it, c);               // moments count of t + 1: the next sweep reads it
    decided();
    if (lane == 0) d2.eta = eta_of(c, t + 2);
  } else if (warp == 3) {
    decided();
    if (lane == 0 && !c.freeze_theta) {
      const U4 r = stream(c.seed, KIND_THETA, 0ull, (uint32_t)(t + 2), 0u);
      d2.u = u01(r.x, r.y);
      d2.lu = hm_log_any_pos(d2.u);
    }
  }
  sync();
  if (!c.freeze_theta) {
    if (warp >= 1) {
      if (lane == 0) theta_consts_part(model, warp - 1, it.thetaP, it.kp);
      if (warp == 1 && lane >= 1 && lane <= nt) {
        const int e = lane - 1, ei = tri_row(e), ej = e - ei * (ei + 1) / 2;
        it.W[e] = make_W_entry(it, d1, ei, ej);
      }
      if (warp == 3 && lane == 0) it.lp_prop_next = log_prior_full(c, it.thetaP, model);
    } else if (lane == 0) {               // warp 0: taps and acceptance bookkeeping of the decision just taken
      it.T_cur_used = it.T_cur; it.lp_cur_used = it.lp_cur;
      it.T_prop = T_prop; it.log_r = log_r; it.alpha_theta = alpha; it.u_theta = d0.u;
      it.accepted_theta = acc;
      it.theta_prop_n += 1;
      if (acc) { it.theta_acc += 1; it.T_cur = T_prop; it.lp_cur = it.lp_prop; }
      decide_counters(it, tot[0], tot[1], tot[3], tot[4]);
    }
  } else if (warp == 0) {
    if (lane < 8) it.kp.v[lane] = it.kc.v[lane];
    if (lane < dt) it.thetaP[lane] = it.theta[lane];
    if (lane == 0) {
      it.lp_prop_next = it.lp_cur;
      it.accepted_theta = 0;
      it.T_prop = 0.0; it.log_r = 0.0; it.alpha_theta = 0.0; it.u_theta = 0.0;
      it.T_cur_used = it.T_cur; it.lp_cur_used = it.lp_cur;
      decide_counters(it, tot[0], tot[1], tot[3], tot[4]);
    }
  }
  if (warp == 2 && trace_or_null && it.trace_write && lane < dt)
    trace_or_null[(it.trace_rows - 1) * dt + lane] = it.theta[lane];
  if (warp == 3 && lane == 1) it.t = t + 1;
  sync();
  // warp 0 read it.lp_prop (the decided iteration's) during phase C, so the next one is moved in only now; the
  // next reader is the decision of iteration t + 1, at least one block barrier away
  if (warp == 3 && lane == 0) it.lp_prop = it.lp_prop_next;
}
#endif

}  // namespace hm
