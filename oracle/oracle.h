/*
 * oracle.h -- C ABI of the CPU oracle for the plate-level RAM Metropolis-within-Gibbs sampler.
 *
 * TEST INFRASTRUCTURE ONLY.  This tree (oracle/) is the slow, single-threaded, obviously-correct
 * restatement of the method of arXiv 2105.08026 (CUDAHM), written from the paper:
 *   - Metropolis-within-Gibbs cycle                         PAPER.md:103-109 (Eq. 2.4, 2.5)
 *   - robust adaptive Metropolis (RAM) steps 1-3            PAPER.md:129-140 (Eq. 2.6)
 *   - theta Metropolis-Hastings step with the population
 *     log-posterior sum
 *   - thinned latent point process likelihood               PAPER.md:228-236 (Eq. 4.3, 4.4)
 *   - BB1 luminosity PDF, priors, flux noise, detection     PAPER.md:256-333 (Eq. 5.1-5.10), :423-450 (Eq. C.2-C.6)
 * It shares no code, header, table or constant with paper_2105_08026_b200/csrc (the CUDA path).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * load it.  All pointers are HOST pointers.  All arrays are structure-of-arrays:
 * chi[j*N + i] is component j of object i; L is the packed lower triangle, row-major
 * ((0,0),(1,0),(1,1),...), L[k*N + i] is packed entry k of object i.
 *
 * Every function returns 0 on success, a negative code on error (never throws).
 * Parity pins: see tests/test_oracle_*.py; every function below is pinned.
 */
#ifndef CUDAHM_ORACLE_H
#define CUDAHM_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct oracle_sampler oracle_sampler;

enum { ORACLE_OK = 0, ORACLE_E_INVALID = -1, ORACLE_E_STATE = -2, ORACLE_E_UNSUPPORTED = -5 };
/* models: */
enum { ORACLE_M_NORMAL1D = 0, ORACLE_M_THINNED_SCHECHTER1D = 1, ORACLE_M_BINORMAL2D = 2, ORACLE_M_LINREG_ME1D = 3,
       ORACLE_M_BB1_FLUXNOISE1D = 4, /* the paper's case study: BB1 population, flux-dependent noise */
       ORACLE_M_NORMAL3D_KNOWNCOV = 5, /* the normal-normal benchmark: 3-vector latents, known C_pop */
       /* the same model for p = 4, 5, 6 (RAM for general dimension, Eq. 2.6) */
       ORACLE_M_NORMAL4D_KNOWNCOV = 6, ORACLE_M_NORMAL5D_KNOWNCOV = 7, ORACLE_M_NORMAL6D_KNOWNCOV = 8 };
enum { ORACLE_F64 = 0, ORACLE_F32_STATE_F64_REDUCE = 1 };
/* Philox stream kinds */
enum { ORACLE_KIND_PLATE = 0, ORACLE_KIND_THETA = 1 };

typedef struct {
  int32_t  model;               /* ORACLE_M_*                                              */
  int32_t  precision;           /* ORACLE_F64 or ORACLE_F32_STATE_F64_REDUCE               */
  int64_t  n_objects;           /* N                                                       */
  uint64_t seed;                /* Philox key                                              */
  double   target_accept_chi;   /* alpha_* of the plate RAM (paper default 0.4)            */
  double   target_accept_theta; /* alpha_* of the theta RAM                                */
  double   eta_exponent;        /* eta_n = n^(-eta_exponent); paper: 2/3                   */
  double   init_scale_chi;      /* S_1 = init_scale_chi * I (paper: identity)              */
  int32_t  freeze_theta;        /* 1: skip the theta step entirely (theta held fixed)      */
  int32_t  keep_chi_moments;    /* 1: accumulate running mean / M2 of chi after burn-in    */
  /* advanced use */
  int64_t  adapt_until;         /* 0: RAM adaptation never stops ("decays with time"); else eta_n = 0
                                   for iterations t > adapt_until (plate and theta factors frozen from then on)   */
  double   prior_mean[8];       /* user prior on theta, multiplying the model's default (uniform):   */
  double   prior_isd[8];        /* independent normal factors N(prior_mean_j, 1/prior_isd_j^2); isd_j = 0: none    */
  /* sharded populations: this sampler owns objects [object_offset, object_offset + n_objects) of
   * n_objects_total (0 = n_objects); object_offset even (objects draw in pairs) */
  int64_t  object_offset, n_objects_total;
  /* frozen members (properties "which should be held fixed over the course of posterior simulation"):
   * 1 = eta_n of object i uses its OWN update count, n_i = (updates of object i so far) + 2, instead of the global
   * n = t + 1; identical as long as every object is updated in every iteration (reading R3) */
  int32_t  per_object_counter;
  int32_t  pad_;
} oracle_config;

/* Per-iteration taps (all optional: a NULL member is skipped).  Per-object arrays have N entries
 * (chi_prop: p*N, L_new: ntri*N), fp32 values are widened exactly to double. */
typedef struct {
  double* chi_prop;   /* Y = X + S U                      (step 1)   */
  double* pi_cur;     /* log l_i(X) + log f(X;theta)                 */
  double* pi_prop;    /* log l_i(Y) + log f(Y;theta)                 */
  double* alpha;      /* min{1, pi(Y)/pi(X)}              (step 2)   */
  double* u;          /* accept uniform                              */
  int32_t* accepted;  /* 1 iff u < alpha                             */
  double* L_new;      /* S_n                              (step 3)   */
  double* a;          /* log f(X_n; theta)                           */
  double* b;          /* log f(X_n; theta')                          */
  /* scalars of the theta step (always written) */
  double theta_prop[8];
  double S, Delta, T_cur, T_prop, lp_cur, lp_prop, log_r, alpha_theta, u_theta;
  int32_t accepted_theta;
  int32_t pad_;
} oracle_taps;

typedef struct {
  int64_t iterations;          /* Gibbs iterations done (t)                  */
  int64_t chi_accepts;         /* accepted plate proposals, all objects      */
  int64_t chi_proposals;
  int64_t theta_accepts;
  int64_t theta_proposals;
  int64_t nonfinite;           /* proposals whose log target was NaN         */
  int64_t moment_samples;
  int64_t trace_rows;
} oracle_stats;

int  oracle_model_dims(int model, int* p, int* dtheta, int* n_data_cols, int* n_consts);
int  oracle_create(const oracle_config* cfg, oracle_sampler** out);
void oracle_destroy(oracle_sampler* s);
int  oracle_set_data(oracle_sampler* s, const double* const* cols, int n_cols);
int  oracle_set_model_consts(oracle_sampler* s, const double* v, int n);
/* Per-object update mask, N bytes: 1 = object i takes RAM steps 1-3 as usual, 0 = object i is held
 * fixed (chi_i, L_i and its update count untouched, no draws consumed) but still contributes log f(chi_i; theta) and
 * log f(chi_i; theta') to the population sums.  NULL = update everything (the default).  May be changed between
 * iterations.  Taps of a held object: chi_prop = chi, pi_prop = pi_cur, alpha = 0, u = 1, accepted = 0, L_new = L. */
int  oracle_set_update_mask(oracle_sampler* s, const uint8_t* mask_or_null);
/* per-object update counts (N values); set_init zeroes them, set_state(t) sets them all to t */
int  oracle_get_counters(oracle_sampler* s, uint32_t* out);
int  oracle_set_counters(oracle_sampler* s, const uint32_t* in);
int  oracle_set_init(oracle_sampler* s, const double* chi0_or_null, const double* theta0,
                     const double* theta_chol0_or_null);
int  oracle_run(oracle_sampler* s, int64_t n_iter, int64_t burn_in, int32_t thin);
int  oracle_step(oracle_sampler* s, int64_t burn_in, int32_t thin, oracle_taps* taps_or_null);
/* the two halves of oracle_step for a sharded population: totals = {S, Delta, -, n_accept, n_nonfinite} of this shard;
 * oracle_shard_decide takes them summed over all shards (objects are independent given theta) */
int  oracle_shard_sweep(oracle_sampler* s, int64_t burn_in, int32_t thin, double* totals);
int  oracle_shard_decide(oracle_sampler* s, int64_t burn_in, int32_t thin, const double* totals_global);
int  oracle_get_theta_trace(oracle_sampler* s, double* out, int64_t cap_rows, int64_t* n_rows);
int  oracle_get_chi_moments(oracle_sampler* s, double* mean, double* var, int64_t cap_objects,
                            int64_t* n_samples);
int  oracle_get_state(oracle_sampler* s, double* chi, double* L, double* theta, double* L_theta,
                      int64_t* t);
int  oracle_set_state(oracle_sampler* s, const double* chi, const double* L, const double* theta,
                      const double* L_theta, int64_t t);
int  oracle_get_stats(oracle_sampler* s, oracle_stats* out);
int  oracle_theta_only(oracle_sampler* s, const double* theta, double* out);        /* T(theta) */
int  oracle_get_selection_table(oracle_sampler* s, double* xk, double* Wk, int cap, int* n);

/* stateless primitives, exported so that the pins can reach each one separately */
void   oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void   oracle_stream_words(uint64_t seed, int kind, uint64_t obj, uint32_t t, uint32_t d, uint32_t out[4]);
double oracle_uniform_f64(uint64_t seed, int kind, uint64_t obj, uint32_t t, uint32_t d);
void   oracle_normals_f64(uint64_t seed, int kind, uint64_t obj, uint32_t t, int n, double* z);
void   oracle_draws_f32(uint64_t seed, int kind, uint64_t obj, uint32_t t, float* z2, float* u);
/* the p normals and the accept uniform of object i at iteration t (objects draw in pairs: oracle/rng.hpp) */
void   oracle_plate_draws_f64(uint64_t seed, uint64_t i, uint32_t t, int p, double* z, double* u);
void   oracle_plate_draws_f32(uint64_t seed, uint64_t i, uint32_t t, int p, float* z, float* u);
double oracle_loglik(int model, const double* chi, const double* data_i, const double* consts);
double oracle_logpop(int model, const double* chi, const double* data_i, const double* theta,
                     const double* consts);
float  oracle_loglik_f32(int model, const float* chi, const float* data_i, const float* consts);
float  oracle_logpop_f32(int model, const float* chi, const float* data_i, const float* theta,
                         const float* consts);
double oracle_logprior(int model, const double* theta);
void   oracle_ram_update(int p, const double* L_packed, const double* z, double c, double* L_out);
void   oracle_gauss_legendre(int n, double a, double b, double* x, double* w);
/* M4: log C(beta, u, l) of PAPER.md:429 (Eq. C.3); the selection integral (Eq. 4.4 denominator) as the plain
 * 1,024 x 512 tensor-product cubature, nothing tabulated.  consts = {sigma_0, alpha, x_lo, x_hi, r_min, r_max, F_th} */
double oracle_bb1_log_norm(double beta, double l, double u);
double oracle_bb1_selection_integral_2d(const double* theta, const double* consts);
double oracle_sum(const double* v, int64_t n);

#ifdef __cplusplus
}
#endif
#endif
