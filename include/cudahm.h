/*
 * cudahm.h -- C ABI of the B200-native plate-level RAM Metropolis-within-Gibbs sampler.
 *
 * What it computes (citations are /root/reference/PAPER.md line numbers, arXiv 2105.08026):
 *   The Metropolis-within-Gibbs cycle of Eq. 2.4-2.5 for a single-plate
 *   hierarchical model (Eq. 2.3).  Per Gibbs iteration t, for every object i:
 *     1. propose  chi' = chi_i + L_i z,  z ~ N(0, I_p)                   (RAM step 1)
 *     2. accept with probability alpha = min{1, pi(chi')/pi(chi_i)},
 *        pi = l_i(.) f(.; theta)                                         (RAM step 2)
 *     3. L_i <- chol(L_i (I + eta_n (alpha - alpha_*) z z^T/|z|^2) L_i^T),
 *        eta_n = n^(-2/3)                                                (RAM step 3, Eq. 2.6)
 *   fused, in the same pass, with the population sums  S = sum_i log f(chi_i; theta)  and
 *   Delta = sum_i [log f(chi_i; theta') - log f(chi_i; theta)]  that the Metropolis-Hastings step
 *   on theta consumes, then the theta decision itself (RAM on theta), running
 *   chi moments and a thinned theta trace.  Models are compiled in (the counterpart of the two
 *   user functions of PAPER.md:144, :391); their definitions are in DESIGN.md section 3.
 *
 * Conventions
 *   - Every function returns a CUDAHM_* status (0 = OK) and never throws; cudahm_last_error()
 *     returns a message for the last failure on that handle (or the global one if the handle is NULL).
 *   - DEVICE MEMORY IS OWNED BY THE CALLER: allocate cudahm_workspace_bytes(cfg) bytes (256-byte
 *     aligned), pass it to cudahm_create; the library sub-allocates all of its state there and never
 *     allocates device memory on the hot path.  The workspace must outlive the handle.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All device work
 *     is enqueued on it.  cudahm_run returns once the work is enqueued (THETA_DEVICE_TAIL, THETA_GRAPH)
 *     or complete (THETA_HOST); every getter synchronises the stream first.
 *   - "T" below is the state precision: double for CUDAHM_F64, float for CUDAHM_F32_STATE_F64_REDUCE.
 *   - Per-object arrays are structure-of-arrays: chi[j*N + i] = component j of object i; L is the
 *     packed lower triangle row-major ((0,0),(1,0),(1,1)): L[k*N + i] = packed entry k of object i.
 *   - theta, L_theta (packed lower triangle of the theta proposal factor), traces and moments are fp64.
 *   - There is no CPU fallback: without a CUDA device every call that needs one fails with CUDAHM_E_CUDA.
 */
#ifndef CUDAHM_H
#define CUDAHM_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct cudahm_sampler cudahm_sampler;   /* opaque; created/destroyed only by the library */

enum { CUDAHM_OK = 0, CUDAHM_E_INVALID = -1, CUDAHM_E_STATE = -2, CUDAHM_E_CUDA = -3,
       CUDAHM_E_WORKSPACE = -4, CUDAHM_E_UNSUPPORTED = -5, CUDAHM_E_NONFINITE = -6 };

/* compiled-in models: (p, dtheta, data columns, model constants) */
enum { CUDAHM_M_NORMAL1D = 0,            /* (1, 2, {y, sigma}, 0)            theta = (mu, log tau)              */
       CUDAHM_M_THINNED_SCHECHTER1D = 1, /* (1, 3, {Fhat, g=1/(4 pi r^2)}, 6) theta = (alpha, log L*, log A)     */
       CUDAHM_M_BINORMAL2D = 2,          /* (2, 5, {y1, y2, s1, s2}, 0)      theta = (m1, m2, l1, l2, zeta)      */
       CUDAHM_M_LINREG_ME1D = 3,         /* (1, 3, {y, sigma, z}, 0)         theta = (a, b, log tau)            */
       /* the paper's case study: BB1 luminosity PDF (Eq. 5.1 / C.2-C.3) in x = ln L, member
        * likelihood = sampling density of Fhat in F with sigma(F)^2 = sigma_0^2 + (alpha F)^2 (Eq. 5.6, 5.8), prior of
        * Eq. 5.5, selection term -N log I(theta) of Eq. 4.3-4.4 with eta of Eq. 5.10                              */
       CUDAHM_M_BB1_FLUXNOISE1D = 4,     /* (1, 3, {Fhat, g=1/(4 pi r^2)}, 7) theta = (beta, log l, log u)       */
       /* the normal-normal benchmark (Eq. 3.1-3.4): chi_i ~ N3(mu, C_pop), y_ij ~ N(chi_ij, sigma_j^2),
        * C_pop and sigma_j known, uniform hyperprior; p = 3 RAM with the general rank-one Cholesky update            */
       CUDAHM_M_NORMAL3D_KNOWNCOV = 5,   /* (3, 3, {y1, y2, y3}, 9)          theta = mu                         */
       /* the same normal-normal model with p-vector latents, p = 4, 5, 6: RAM for general dimension (Eq. 2.6, PAPER.md:129-140,
        * is stated for any p; section 3 is its p = 3 instance).  (p, p, {y1..yp}, p + p(p+1)/2), theta = mu.  F64 only, 256-thread blocks */
       CUDAHM_M_NORMAL4D_KNOWNCOV = 6, CUDAHM_M_NORMAL5D_KNOWNCOV = 7, CUDAHM_M_NORMAL6D_KNOWNCOV = 8 };
enum { CUDAHM_F64 = 0, CUDAHM_F32_STATE_F64_REDUCE = 1 };
/* where the theta Metropolis-Hastings step runs (PAPER.md:142 puts it on the host) */
enum { CUDAHM_THETA_HOST = 0,         /* one sweep launch + one sync per iteration; theta step in host C++     */
       CUDAHM_THETA_GRAPH = 1,        /* {sweep kernel, 1-block tail kernel} per iteration, CUDA-Graph batches */
       CUDAHM_THETA_DEVICE_TAIL = 2 };/* one persistent cooperative kernel, one grid barrier per iteration     */

/* cudahm_config.flags: THETA_DEVICE_TAIL keeps a population that fits in shared memory on chip for the whole run
 * (fp64, p = 1 models); this flag forces the HBM-streaming persistent kernel instead. */
enum { CUDAHM_FLAG_STREAMING_ONLY = 1,
       CUDAHM_FLAG_TMA_STAGING = 2 };  /* stream through TMA-staged shared-memory tiles (stream_tma.cuh) instead of
                                          plain vector loads; measured slower on C3 / C4, kept as an option          */
/* bits 8-15 of flags: the streaming persistent kernel makes the plate draws (U_n ~ q) of each thread's
 * first n steps of iteration t + 1 while the exchange and the theta step of iteration t are in flight; 0 in these
 * bits = automatic, CUDAHM_FLAG_STAGE_STEPS(n) = exactly n (n = 0: off), clipped to what fits in shared memory.
 * The chain is the same bit for bit whatever n is.                                                                */
/* the streaming persistent kernel prefetches the columns of a thread's next step into L2 while it computes the current
 * one, by default when state + data exceed the L2 cache (they then stream from HBM every iteration); these two force it */
#define CUDAHM_FLAG_PREFETCH_OFF 4
#define CUDAHM_FLAG_PREFETCH_ON 8
/* bracket every cudahm_run with a pair of CUDA events so that cudahm_stats.last_run_ms is filled.  Off by default: the two
 * event records cost about 5 us of device front-end time per run, as much as one Gibbs iteration at N = 3e5. */
#define CUDAHM_FLAG_TIME_RUNS 16
#define CUDAHM_FLAG_STAGE_STEPS_MASK 0xff00
#define CUDAHM_FLAG_STAGE_STEPS(n) ((((n) + 1) << 8) & CUDAHM_FLAG_STAGE_STEPS_MASK)

typedef struct {
  uint32_t struct_size;          /* sizeof(cudahm_config), checked                                          */
  int32_t  model;                /* CUDAHM_M_*                                                              */
  int32_t  precision;            /* CUDAHM_F64 | CUDAHM_F32_STATE_F64_REDUCE                                */
  int32_t  theta_mode;           /* CUDAHM_THETA_*                                                          */
  int64_t  n_objects;            /* N >= 0                                                                  */
  int32_t  p, dtheta, n_data_cols; /* must match the compiled-in model, else CUDAHM_E_INVALID               */
  int32_t  freeze_theta;         /* 1: skip the theta step (theta held fixed)                               */
  uint64_t seed;                 /* Philox4x32-10 key                                                       */
  double   target_accept_chi;    /* alpha_* of the plate RAM; paper default 0.4              */
  double   target_accept_theta;  /* alpha_* of the theta RAM (paper-silent; reading R7)           */
  double   eta_exponent;         /* eta_n = n^(-eta_exponent); paper: 2/3                    */
  double   init_scale_chi;       /* S_1 = init_scale_chi * I; paper: identity                */
  int32_t  keep_chi_moments;     /* 1: running mean / variance of every chi component after burn-in         */
  int32_t  block_threads;        /* 0 = default; else 256, 512 or 1024                                      */
  int32_t  blocks_per_sm;        /* 0 = as many as fit; else an upper limit                                 */
  int32_t  flags;                /* 0, or CUDAHM_FLAG_* ORed                                                */
  int64_t  max_trace_rows;       /* capacity of the on-device thinned theta trace (rows of dtheta doubles);
                                    0 = keep no trace                                                        */
  /* advanced use.  Precisely measured predictors are read-only data columns (M3's z, the g
   * column of M1 / M4), which is what PAPER.md:397-399 asks users to arrange by overriding the default kernels.  */
  int64_t  adapt_until;          /* 0: the RAM adaptation never stops (it "decays with time"); else
                                    eta_n = 0 for t > adapt_until: plate and theta proposal factors are frozen  */
  double   prior_mean[8];        /* user prior on theta multiplying the model's default (the default */
  double   prior_isd[8];         /* is uniform and can be overridden): independent normal factors
                                    N(prior_mean[j], 1/prior_isd[j]^2) on theta[j]; prior_isd[j] = 0: no factor   */
  /* sharding over several samplers / GPUs (cudahm_shard_sweep / cudahm_shard_decide below): this handle owns the
   * objects [object_offset, object_offset + n_objects) of a population of n_objects_total                          */
  int64_t  object_offset;        /* even, >= 0: global index of this handle's first object (keys its Philox streams) */
  int64_t  n_objects_total;      /* 0 = n_objects (not sharded)                                                    */
  /* frozen members (member properties "which should be held fixed over the course of posterior
   * simulation").  Either switch selects the HOLD variants of the streaming kernels (not the on-chip kernel, no staged
   * draws / TMA); as-built extra state: 1 byte (mask) and 4 bytes (counter) per object, read and written every iteration. */
  int32_t  update_mask;          /* 1: reserve a per-object update mask (cudahm_set_update_mask); all ones until set    */
  int32_t  per_object_counter;   /* 1: eta_n of object i uses ITS OWN update count, n_i = count_i + 2, instead of the
                                    global n = t + 1 (identical while every object is updated in every iteration)  */
} cudahm_config;

typedef struct {
  int64_t iterations;            /* Gibbs iterations done (t)                                               */
  int64_t chi_accepts;           /* accepted plate proposals over all objects and iterations                */
  int64_t chi_proposals;
  int64_t theta_accepts;
  int64_t theta_proposals;
  int64_t nonfinite;             /* plate proposals whose log target ratio was NaN (rejected, alpha = 0)    */
  int64_t moment_samples;        /* post-burn-in iterations accumulated into the chi moments                */
  int64_t trace_rows;
  int64_t gpu_launches;          /* kernels launched by this handle so far                                  */
  int32_t grid_blocks, block_threads;   /* launch configuration of the sweep                               */
  double  last_run_ms;           /* device time of the last cudahm_run (needs CUDAHM_FLAG_TIME_RUNS; else 0)  */
  int32_t stage_steps;           /* streaming persistent kernel: steps of plate draws staged ahead per thread */
  int32_t l2_prefetch;           /* ... 1: it prefetches the next step's columns into L2 (0 for the on-chip kernel) */
  int32_t dedicated_tail;        /* 1: the streaming kernel with dedicated tail warps (k_persistent_dt) runs             */
  int32_t graph_launches;        /* persistent-kernel launches submitted through the handle's one-node CUDA graph (every
                                    cudahm_run in THETA_DEVICE_TAIL mode after the handle's first; 0 = direct launches only) */
} cudahm_stats;

/* Per-iteration taps of cudahm_debug_step; HOST pointers, each may be NULL.  Values are widened to double. */
typedef struct {
  double* chi_prop;    /* p*N    chi' = chi + L z                                                           */
  double* pi_cur;      /* N      log l_i(chi) + log f(chi; theta)                                           */
  double* pi_prop;     /* N      same at chi'                                                               */
  double* alpha;       /* N      min{1, pi(chi')/pi(chi)}                                                   */
  double* u;           /* N      accept uniform                                                             */
  int32_t* accepted;   /* N      1 iff u < alpha                                                            */
  double* L_new;       /* ntri*N updated factor                                                             */
  double* a;           /* N      log f(chi_new; theta)                                                      */
  double* b;           /* N      log f(chi_new; theta')                                                     */
  double  theta_prop[8];
  double  S, Delta, T_cur, T_prop, lp_cur, lp_prop, log_r, alpha_theta, u_theta;
  int32_t accepted_theta;
  int32_t pad_;
} cudahm_taps;

/* Model dimensions: (p, dtheta, n_data_cols, n_consts).  CUDAHM_E_INVALID for an unknown model. */
int cudahm_model_dims(int model, int* p, int* dtheta, int* n_data_cols, int* n_consts);

/* Bytes of device workspace the configuration needs (0 if cfg is invalid). */
size_t cudahm_workspace_bytes(const cudahm_config* cfg);

/* Create a sampler inside the caller's device workspace.  CUDAHM_E_WORKSPACE if `bytes` is too small or the
 * pointer is not 256-byte aligned; CUDAHM_E_UNSUPPORTED for a (model, precision) pair that is not compiled in
 * (compiled in: every model in F64; NORMAL1D and LINREG_ME1D in F32_STATE_F64_REDUCE). */
int cudahm_create(const cudahm_config* cfg, void* dev_workspace, size_t bytes, void* cuda_stream,
                  cudahm_sampler** out);
void cudahm_destroy(cudahm_sampler* s);

/* Copy the n_cols data columns (arrays of N values of type T, host or device) into the workspace; the caller's
 * buffers may be freed afterwards.  Member likelihoods l_i are built from them. */
int cudahm_set_data(cudahm_sampler* s, const void* const* cols, int n_cols, int cols_on_device);

/* Model constants (host doubles).  THINNED_SCHECHTER1D: {F_lim, sigma_F, x_lo, x_hi, r_min, r_max};
 * BB1_FLUXNOISE1D: {sigma_0, alpha, x_lo, x_hi, r_min, r_max, F_th} (Eq. 5.8-5.10); both build the 1,024-point
 * selection-integral table (Eq. 4.4 denominator).  NORMAL3D_KNOWNCOV: {sigma_1, sigma_2, sigma_3, C11, C21,
 * C22, C31, C32, C33} (packed lower triangle of C_pop, Eq. 3.3); NORMAL4D .. 6D likewise: {sigma_1..p, packed lower triangle
 * of C_pop row-major}; CUDAHM_E_INVALID unless sigma_j > 0 and C_pop is positive definite.  Other models take n = 0. */
int cudahm_set_model_consts(cudahm_sampler* s, const double* v, int n);

/* Initial state: chi0 (p*N values of type T, host or device per chi0_on_device; NULL = the model's default
 * X_1, reading R6), theta0 (dtheta host doubles), theta_chol0 (packed lower triangle, host doubles;
 * NULL = 0.1 * I).  Resets t = 0, L_i = init_scale_chi * I, the trace, the moments and the counters.
 * CUDAHM_E_STATE before set_data (and set_model_consts where the model has constants); CUDAHM_E_NONFINITE if theta0 has
 * zero prior density or a non-finite theta-only term (the chain needs pi(X_1) > 0; set_state likewise). */
int cudahm_set_init(cudahm_sampler* s, const void* chi0_or_null, int chi0_on_device, const double* theta0,
                    const double* theta_chol0_or_null);

/* Per-object update mask (needs cfg.update_mask): N bytes, host or device; 1 = object i takes RAM steps 1-3 as usual,
 * 0 = object i is held fixed -- chi_i, L_i and its update count stay bit for bit -- but still contributes log f(chi_i; theta)
 * and log f(chi_i; theta') to the population sums.  NULL = update everything again.  May be changed between runs; copied.
 * Taps of a held object: chi_prop = chi, pi_prop = pi_cur, alpha = 0, u = 1, accepted = 0, L_new = L.  chi_proposals counts
 * updated objects only.  CUDAHM_E_STATE without cfg.update_mask, CUDAHM_E_UNSUPPORTED on a sharded handle. */
int cudahm_set_update_mask(cudahm_sampler* s, const uint8_t* mask_or_null, int mask_on_device);
/* Per-object update counts (needs cfg.per_object_counter), N host values.  set_init zeroes them, set_state(t) sets them
 * all to t (as if every object had been updated in every iteration so far); set_counters overrides. */
int cudahm_get_counters(cudahm_sampler* s, uint32_t* out);
int cudahm_set_counters(cudahm_sampler* s, const uint32_t* in);

/* Run n_iter more Gibbs iterations (resumable: continues from the current iteration index t).  Moments are
 * accumulated for t > burn_in, the trace takes theta whenever t > burn_in and (t - burn_in) % thin == 0.
 * CUDAHM_E_INVALID if the trace would overflow max_trace_rows (max_trace_rows == 0 keeps no trace at all).
 * Asynchronous: the work is queued on the handle's stream, nothing is read back.  May be called with any device current
 * (the device that was current at cudahm_create is made current for the duration of the call); every other call expects
 * the handle's device to be current.  In THETA_DEVICE_TAIL mode a handle's first run is submitted as a direct cooperative
 * launch, later ones through a one-node CUDA graph whose parameters are updated in place (cudahm_stats.graph_launches). */
int cudahm_run(cudahm_sampler* s, int64_t n_iter, int64_t burn_in, int32_t thin);

/* Sharded populations: objects are conditionally independent given theta (Eq. 2.4), so a
 * population splits by object range over several handles (one per GPU); theta, L_theta and the theta Philox stream are
 * replicated, and the only exchange per Gibbs iteration is the sum of the handles' totals.  THETA_HOST handles only
 * (CUDAHM_E_UNSUPPORTED otherwise).
 *   cudahm_shard_sweep:  one fused sweep over this handle's objects; totals[5] (host doubles) receives
 *                        {S, Delta, Tq, n_accept, n_nonfinite} of THIS shard.  S, Delta, n_accept, n_nonfinite are to be
 *                        summed over the shards (in a fixed order, so every rank holds the same bits); Tq (the selection
 *                        sum of M1 / M4) is computed in full by every handle and must NOT be summed.
 *   cudahm_shard_decide: the theta step of the iteration just swept from the GLOBAL totals, identical on every handle;
 *                        prepares the next iteration.
 * A handle with object_offset = 0 and n_objects_total = n_objects reproduces cudahm_run(THETA_HOST) bit for bit. */
int cudahm_shard_sweep(cudahm_sampler* s, int64_t burn_in, int32_t thin, double* totals);
int cudahm_shard_decide(cudahm_sampler* s, int64_t burn_in, int32_t thin, const double* totals_global);
/* The fixed-order (rank-order) sum of the shards' totals: out[5] = {sum S, sum Delta, Tq of rank 0, sum n_accept,
 * sum n_nonfinite} from totals_by_rank[n_ranks][5] (host doubles).  Pure host arithmetic, no device needed: every rank
 * that calls it on the same gathered array holds the same bits. */
int cudahm_shard_combine(const double* totals_by_rank, int n_ranks, double* out);
/* The same two halves without a host bounce between them, for an exchange that runs on the device (NCCL all-gather on the
 * sampler's stream): shard_sweep_device leaves this shard's five totals in the caller's DEVICE buffer totals_dev[5]
 * (enqueued, no synchronisation); shard_decide_gathered takes the DEVICE array gathered_dev[n_ranks][5] in rank order,
 * reads it back once (40 n_ranks bytes), combines it with cudahm_shard_combine's rule and takes the theta step. */
int cudahm_shard_sweep_device(cudahm_sampler* s, int64_t burn_in, int32_t thin, void* totals_dev);
int cudahm_shard_decide_gathered(cudahm_sampler* s, int64_t burn_in, int32_t thin, const void* gathered_dev, int n_ranks);

/* One iteration through the non-persistent sweep + tail kernels with per-object taps (test instrument). */
int cudahm_debug_step(cudahm_sampler* s, int64_t burn_in, int32_t thin, cudahm_taps* taps);

/* cudahm_debug_step for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses
 * that forbid it): identical kernels and taps, but the per-object tap scratch -- (p + p(p+1)/2 + 6) doubles and one int per
 * object, which cudahm_debug_step cudaMallocs and frees on every call -- lives in ONE file-scope device array of
 * CUDAHM_NOALLOC_SCRATCH_BYTES that every GPU loading the library holds until the process exits.  The call allocates no
 * device memory (no cudaMalloc / cudaFree / allocating library routine).  CUDAHM_E_WORKSPACE, with nothing touched, if the
 * handle needs more than the array holds (cudahm_debug_step_noalloc_bytes(s) says how much: p = 1 fits about 61,600
 * objects, p = 2 45,500, p = 6 15,600).  Every call on a device shares the array, which keeps the previous call's contents: the range
 * a call uses is cleared before its kernels run, and calls that OVERLAP on the GPU (other streams, other host threads) race
 * -- serialise them.  The handle's device must be current, as for every other call. */
#define CUDAHM_NOALLOC_SCRATCH_BYTES (4u << 20)
int cudahm_debug_step_noalloc(cudahm_sampler* s, int64_t burn_in, int32_t thin, cudahm_taps* taps);
size_t cudahm_debug_step_noalloc_bytes(const cudahm_sampler* s);

/* Results.  Both calls queue their transfers on the handle's stream behind the runs already submitted and synchronise that
 * stream once before they return; the row / sample counts come from host-side mirrors (functions of the (t, burn_in, thin)
 * history), so nothing else is read back.  Host buffers may be pageable or pinned (pinned ones move at PCIe speed).
 * out: row-major n_rows x dtheta host doubles.  out == NULL just reports n_rows, without synchronising. */
int cudahm_get_theta_trace(cudahm_sampler* s, double* out, int64_t cap_rows, int64_t* n_rows);
/* mean, var: p*N host doubles (SoA); var is the sample variance (divisor n_samples - 1). */
int cudahm_get_chi_moments(cudahm_sampler* s, double* mean, double* var, int64_t cap_objects, int64_t* n_samples);
int cudahm_get_stats(cudahm_sampler* s, cudahm_stats* out);
/* chi, L: host arrays of T (p*N, ntri*N); theta, L_theta: host doubles; any pointer may be NULL. */
int cudahm_get_state(cudahm_sampler* s, void* chi, void* L, double* theta, double* L_theta, int64_t* t);
int cudahm_set_state(cudahm_sampler* s, const void* chi, const void* L, const double* theta,
                     const double* L_theta, int64_t t);
/* Block until everything enqueued on the sampler's stream is done; reports asynchronous CUDA errors. */
int cudahm_sync(cudahm_sampler* s);
const char* cudahm_last_error(const cudahm_sampler* s_or_null);

#ifdef __cplusplus
}
#endif
#endif
