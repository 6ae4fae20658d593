// cudahm.cu -- host side of the C ABI declared in include/cudahm.h: argument checks, workspace layout,
// kernel dispatch and the three theta-step drivers (device tail / CUDA graph / host).  No CPU fallback:
// every step of the path runs in the kernels of kernels.cuh.
#include "cudahm.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <utility>
#include <vector>

#include "kernel_sets.h"
#include "tail_kernels.cuh"
#include "resident_cfg.h"

using namespace hm;

namespace {

thread_local std::string g_err;

struct Layout {
  size_t chi, L, data, mom_mean, mom_M2, mom_var, slots, mbox, blk_cnt, iter, trace, totals, qx, qex, qW, mask, cnt, total;
};

constexpr int MAX_BLOCKS = 148 * 8 * 2;   // upper bound on the grid (slots capacity)
constexpr int MAX_PGRID = 320;            // upper bound on the persistent grid (mailboxes grow with its square)
constexpr int STAGE_STEPS_AUTO = 2;       // staged steps of plate draws when the flags do not say
constexpr size_t STAGE_MAX_SMEM = 192 * 1024;   // dynamic shared memory k_persistent may ask for

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// kernels of one (model, precision, block size): the per-model translation units inst_*.cu hold the instantiations
bool pick_kernels(int model, int precision, int block, KernelSet* k, ResidentSet* r) {
  switch (model) {
    case M_NORMAL1D:            return kernels_normal1d(precision, block, k, r);
    case M_THINNED_SCHECHTER1D: return kernels_thinned_schechter1d(precision, block, k, r);
    case M_BINORMAL2D:          return kernels_binormal2d(precision, block, k, r);
    case M_LINREG_ME1D:         return kernels_linreg_me1d(precision, block, k, r);
    case M_BB1_FLUXNOISE1D:     return kernels_bb1_fluxnoise1d(precision, block, k, r);
    case M_NORMAL3D_KNOWNCOV:   return kernels_normal3d_knowncov(precision, block, k, r);
    case M_NORMAL4D_KNOWNCOV:   return kernels_normal4d_knowncov(precision, block, k, r);
    case M_NORMAL5D_KNOWNCOV:   return kernels_normal5d_knowncov(precision, block, k, r);
    case M_NORMAL6D_KNOWNCOV:   return kernels_normal6d_knowncov(precision, block, k, r);
  }
  return false;
}

}  // namespace

struct cudahm_sampler {
  cudahm_config cfg{};
  Params P{};
  Layout lay{};
  KernelSet ks{};
  cudaStream_t stream = nullptr;
  char* ws = nullptr;
  int p = 0, dtheta = 0, ncols = 0, nconsts = 0, ntri = 0, ntri_theta = 0;
  size_t tsize = 8;
  bool have_data = false, have_consts = false, have_init = false;
  int num_sms = 0, grid = 1, block = 512, vec = 2;
  long long t_done = 0;             // iterations completed (host mirror)
  bool hold = false;                // frozen-member kernel variants (update mask and / or per-object counter)
  long long n_active = 0;           // objects the mask lets update (N without a mask)
  long long h_proposals = 0;        // plate proposals made so far (host mirror: iterations x updated objects)
  long long h_trace_rows = 0;       // host mirrors of Iter::trace_rows / mom_count: pure functions of the (t, burn_in, thin)
  long long h_mom_count = 0;        // history, so cudahm_run never has to read the device before it launches
  long long launches = 0;
  Iter* h_iter = nullptr;           // pinned host copy of the iteration state
  double* h_totals = nullptr;       // pinned
  bool host_iter_valid = false;     // THETA_HOST: h_iter is authoritative between runs
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  bool timed = false;
  unsigned epoch = 1;               // next mailbox epoch of the persistent kernel
  const void* res_kernel = nullptr; // on-chip persistent kernel (resident.cuh) when the population fits, else NULL
  int res_R = 0, res_OB = 0, res_threads = 0; size_t res_smem = 0;
  int sweep_grid = 1, sweep_block = 512;   // launch shape of k_sweep (THETA_GRAPH / HOST / debug_step)
  int tma_stages = 0; size_t tma_smem = 0;   // > 0: the streaming persistent kernel is k_persistent_tma
  bool ahead = false;                        // run k_persistent<.., AHEAD = true>
  bool dt = false;                           // run k_persistent_dt (dedicated tail warps)
  int prefetch = 0;                          // ... with L2 prefetch of the next step's columns
  int n_stage = 0; size_t stage_smem = 0;    // k_persistent: steps of plate draws staged in shared memory ahead of the sweep
  double h_lp_prop_before = 0.0;    // log prior at theta' of the iteration debug_step is about to decide
  // CUDA-graph cache (THETA_GRAPH)
  cudaGraphExec_t pg_exec = nullptr;          // one-node graph of the persistent kernel (launch_persistent)
  cudaGraph_t pg_graph = nullptr;             // ... the graph pg_node lives in: kept as long as pg_exec (the in-place update names the node)
  cudaGraphNode_t pg_node = nullptr;
  int pg_graph_launches = 0;                  // launches that went out through pg_exec (cudahm_stats.graph_launches)
  int device = 0;                             // the device that was current at cudahm_create (owns workspace and stream)
  const void* pg_fn = nullptr;
  bool pg_broken = false;
  long long pg_launches = 0;
  cudaGraphExec_t gexec = nullptr;
  long long g_burn = -1; int g_thin = -1; int g_iters = 0;
  std::string err;
};

namespace {

int fail(cudahm_sampler* s, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  if (s) s->err = buf;
  return code;
}

// the captured k_sweep / k_tail nodes of THETA_GRAPH hold Params BY VALUE (model constants, pointers, prior): anything
// that changes them, or rewinds the chain, drops the cached executable graph so the next run captures afresh
void drop_persistent_graph(cudahm_sampler* s) {
  if (s->pg_exec) { cudaGraphExecDestroy(s->pg_exec); s->pg_exec = nullptr; }
  if (s->pg_graph) { cudaGraphDestroy(s->pg_graph); s->pg_graph = nullptr; }
  s->pg_node = nullptr; s->pg_fn = nullptr;
}

void invalidate_graph(cudahm_sampler* s) {
  if (s->gexec) { cudaGraphExecDestroy(s->gexec); s->gexec = nullptr; }
  s->g_burn = -1; s->g_thin = -1; s->g_iters = 0;
}

#define CU_TRY(s, call)                                                                      \
  do {                                                                                       \
    cudaError_t e_ = (call);                                                                 \
    if (e_ != cudaSuccess) return fail(s, CUDAHM_E_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the FUNCTION (per device), not to a handle: keep a process-wide
// maximum per (device, function) and only ever raise it, so that two handles of one model with different N cannot lower
// each other's limit between create and launch.
cudaError_t ensure_dyn_smem(const void* fn, size_t bytes) {
  static std::mutex mu;
  static std::map<std::pair<int, const void*>, size_t> have;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(mu);
  size_t& cur = have[{dev, fn}];
  if (bytes <= cur) return cudaSuccess;
  e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  if (e == cudaSuccess) cur = bytes;
  return e;
}

// rows the thinned trace gains / post-burn-in iterations the moments gain over iterations (t0, t1]
long long trace_rows_between(long long t0, long long t1, long long burn_in, long long thin) {
  const long long lo = std::max(t0, burn_in);
  return t1 > lo ? (t1 - burn_in) / thin - (lo - burn_in) / thin : 0;
}
long long moment_samples_between(long long t0, long long t1, long long burn_in) {
  const long long lo = std::max(t0, burn_in);
  return t1 > lo ? t1 - lo : 0;
}

bool valid_config(const cudahm_config* c, int* p, int* dt, int* nc, int* nk) {
  if (!c || c->struct_size != sizeof(cudahm_config)) return false;
  if (!model_dims(c->model, p, dt, nc, nk)) return false;
  if (c->p != *p || c->dtheta != *dt || c->n_data_cols != *nc) return false;
  if (c->n_objects < 0 || c->max_trace_rows < 0 || (c->flags & ~(CUDAHM_FLAG_STREAMING_ONLY | CUDAHM_FLAG_TMA_STAGING | CUDAHM_FLAG_STAGE_STEPS_MASK | CUDAHM_FLAG_PREFETCH_OFF | CUDAHM_FLAG_TIME_RUNS |
                                                              CUDAHM_FLAG_PREFETCH_ON)) != 0) return false;
  if (c->precision != CUDAHM_F64 && c->precision != CUDAHM_F32_STATE_F64_REDUCE) return false;
  if (c->theta_mode < CUDAHM_THETA_HOST || c->theta_mode > CUDAHM_THETA_DEVICE_TAIL) return false;
  if (!(c->target_accept_chi > 0.0 && c->target_accept_chi < 1.0)) return false;
  if (!(c->target_accept_theta > 0.0 && c->target_accept_theta < 1.0)) return false;
  if (!(c->eta_exponent > 0.0 && c->eta_exponent <= 1.0) || !(c->init_scale_chi > 0.0)) return false;
  if (c->block_threads != 0 && c->block_threads != 256 && c->block_threads != 512 && c->block_threads != 1024)
    return false;
  if (c->blocks_per_sm < 0 || c->adapt_until < 0) return false;
  if (c->object_offset < 0 || (c->object_offset & 1) || c->n_objects_total < 0) return false;
  if ((c->update_mask | c->per_object_counter) & ~1) return false;
  if (c->n_objects_total != 0 && c->object_offset + c->n_objects > c->n_objects_total) return false;
  for (int j = 0; j < 8; ++j)
    if (!(c->prior_isd[j] >= 0.0) || !std::isfinite(c->prior_isd[j]) || !std::isfinite(c->prior_mean[j])) return false;
  return true;
}

Layout make_layout(const cudahm_config& c, int p, int ncols, int dtheta) {
  const size_t ts = c.precision == CUDAHM_F64 ? 8 : 4;
  const size_t Npad = (size_t)((c.n_objects + 31) / 32 * 32);
  const int ntri = p * (p + 1) / 2;
  Layout l{};
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
  l.chi = take((size_t)p * Npad * ts);
  l.L = take((size_t)ntri * Npad * ts);
  l.data = take((size_t)ncols * Npad * ts);
  const size_t mom = c.keep_chi_moments ? (size_t)p * Npad * 8 : 0;
  l.mom_mean = take(mom); l.mom_M2 = take(mom); l.mom_var = take(mom);
  l.slots = take((size_t)MAX_BLOCKS * NPART * 8);
  l.mbox = take((size_t)2 * MAX_PGRID * MAX_PGRID * 2 * MBOX_NV * 8);
  l.blk_cnt = take((size_t)MAX_BLOCKS * 2 * 8);
  l.iter = take(sizeof(Iter));
  l.trace = take((size_t)c.max_trace_rows * dtheta * 8);
  l.totals = take(NPART * 8);
  l.qx = take(NQUAD * 8); l.qex = take(NQUAD * 8); l.qW = take(NQUAD * 8);
  l.mask = take(c.update_mask ? Npad : 0);
  l.cnt = take(c.per_object_counter ? Npad * 4 : 0);
  l.total = o;
  return l;
}

}  // namespace

// ----------------------------------------------------------------------------------------------------
extern "C" int cudahm_model_dims(int model, int* p, int* dtheta, int* n_data_cols, int* n_consts) {
  int a, b, c, d;
  if (!model_dims(model, &a, &b, &c, &d)) return fail(nullptr, CUDAHM_E_INVALID, "unknown model %d", model);
  if (p) *p = a;
  if (dtheta) *dtheta = b;
  if (n_data_cols) *n_data_cols = c;
  if (n_consts) *n_consts = d;
  return CUDAHM_OK;
}

extern "C" size_t cudahm_workspace_bytes(const cudahm_config* cfg) {
  int p, dt, nc, nk;
  if (!valid_config(cfg, &p, &dt, &nc, &nk)) return 0;
  return make_layout(*cfg, p, nc, dt).total;
}

extern "C" const char* cudahm_last_error(const cudahm_sampler* s) { return s ? s->err.c_str() : g_err.c_str(); }

extern "C" int cudahm_create(const cudahm_config* cfg, void* dev_workspace, size_t bytes, void* cuda_stream,
                             cudahm_sampler** out) {
  if (!out) return fail(nullptr, CUDAHM_E_INVALID, "out is NULL");
  *out = nullptr;
  int p, dt, nc, nk;
  if (!valid_config(cfg, &p, &dt, &nc, &nk)) return fail(nullptr, CUDAHM_E_INVALID, "invalid cudahm_config");
  // default block: 512 threads; a population too small to give every SM a 512-thread block of 16-byte vectors takes
  // 256-thread blocks instead (twice the SMs at work: the small configs are latency-bound, not bandwidth-bound)
  int block = cfg->block_threads ? cfg->block_threads : 512;
  if (!cfg->block_threads && p >= 4) block = 256;     // two objects of p (p + 5) / 2 doubles each per thread: 255 registers
  else if (!cfg->block_threads) {
    const long long vec = cfg->precision == CUDAHM_F64 ? 2 : 4;
    int dev0 = 0, sms0 = 0;
    if (cudaGetDevice(&dev0) == cudaSuccess) cudaDeviceGetAttribute(&sms0, cudaDevAttrMultiProcessorCount, dev0);
    if ((cfg->n_objects + vec * 512 - 1) / (vec * 512) < (sms0 > 0 ? sms0 : 148)) block = 256;
  }
  if (cfg->update_mask && cfg->n_objects_total != 0 && cfg->n_objects_total != cfg->n_objects)
    return fail(nullptr, CUDAHM_E_UNSUPPORTED, "an update mask on a sharded handle is not supported");
  KernelSet ks;
  ResidentSet rs;
  if (!pick_kernels(cfg->model, cfg->precision, block, &ks, &rs))
    return fail(nullptr, CUDAHM_E_UNSUPPORTED, "model %d is not compiled in for precision %d", cfg->model, cfg->precision);
  const Layout lay = make_layout(*cfg, p, nc, dt);
  if (!dev_workspace || bytes < lay.total || ((uintptr_t)dev_workspace & 255u))
    return fail(nullptr, CUDAHM_E_WORKSPACE, "workspace must be 256-byte aligned and >= %zu bytes (got %zu)", lay.total, bytes);
  int dev = 0, sms = 0, coop = 0;
  CU_TRY(nullptr, cudaGetDevice(&dev));
  CU_TRY(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  CU_TRY(nullptr, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
  if (!coop) return fail(nullptr, CUDAHM_E_CUDA, "device does not support cooperative launches");

  cudahm_sampler* s = new cudahm_sampler();
  s->cfg = *cfg; s->lay = lay; s->ks = ks; s->stream = (cudaStream_t)cuda_stream; s->ws = (char*)dev_workspace; s->device = dev;
  s->p = p; s->dtheta = dt; s->ncols = nc; s->nconsts = nk; s->ntri = p * (p + 1) / 2; s->ntri_theta = dt * (dt + 1) / 2;
  s->tsize = cfg->precision == CUDAHM_F64 ? 8 : 4;
  s->vec = cfg->precision == CUDAHM_F64 ? 2 : 4;
  s->num_sms = sms; s->block = block;
  s->have_consts = (nk == 0);
  s->hold = cfg->update_mask || cfg->per_object_counter;
  s->n_active = cfg->n_objects_total ? cfg->n_objects_total : cfg->n_objects;

  int per_sm = 0;
  cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ks.persistent, block, 0);
  if (e != cudaSuccess || per_sm < 1) { delete s; return fail(nullptr, CUDAHM_E_CUDA, "occupancy query failed: %s", cudaGetErrorString(e)); }
  if (cfg->blocks_per_sm > 0) per_sm = std::min(per_sm, (int)cfg->blocks_per_sm);
  long long need = (cfg->n_objects + (long long)s->vec * block - 1) / ((long long)s->vec * block);
  s->grid = (int)std::max(1LL, std::min<long long>((long long)sms * per_sm, need));
  s->grid = std::min(s->grid, MAX_BLOCKS);
  if (cfg->theta_mode == CUDAHM_THETA_DEVICE_TAIL && s->grid > MAX_PGRID) s->grid = std::max(1, MAX_PGRID / sms) * sms;
  s->sweep_grid = s->grid; s->sweep_block = block;
  // The AHEAD variant of k_persistent:
  // (i) a state + data set larger than L2 streams from HBM every iteration: the sweep prefetches the columns of its
  //     next step into L2 while it computes the current one.  A set that L2 holds (C3: 72 MB) gains nothing;
  // (ii) the plate draws of each thread's first n_stage steps of iteration t + 1 are made while the exchange and the
  //     theta step of iteration t are in flight (they depend on (seed, object, t) only) and wait in shared memory.
  //     Measured gains: p = 1 out of L2 -13 %, C6 (p = 3, one step) -10 %, C4 -0.5 %; C3 (p = 2: the fp64 draws of
  //     one step take the idle warps as long as the whole exchange) loses 5 % to the plain kernel, which it keeps.
  if (cfg->theta_mode == CUDAHM_THETA_DEVICE_TAIL && cfg->n_objects > 0 && !s->hold) {
    int l2 = 0;
    cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev);
    const size_t set_bytes = (size_t)(p + p * (p + 1) / 2 + nc) * (size_t)cfg->n_objects * s->tsize;
    s->prefetch = (cfg->flags & CUDAHM_FLAG_PREFETCH_ON) ? 1 : (cfg->flags & CUDAHM_FLAG_PREFETCH_OFF) ? 0 : set_bytes > (size_t)l2;
    const long long per_step = (long long)s->vec * block * s->grid;
    const long long steps = (cfg->n_objects + per_step - 1) / per_step;
    const int asked = (cfg->flags & CUDAHM_FLAG_STAGE_STEPS_MASK) >> 8;       // 0 = automatic, else steps + 1
    long long ns = asked ? asked - 1 : (p == 2 && !s->prefetch ? 0 : STAGE_STEPS_AUTO);
    ns = std::min<long long>(std::min(ns, steps), (long long)(STAGE_MAX_SMEM / ks.stage_step_bytes));
    for (; ns > 0; --ns) {
      const size_t bytes = (size_t)ns * ks.stage_step_bytes;
      int fit = 0;
      if (ensure_dyn_smem(ks.persistent_ahead, bytes) == cudaSuccess &&
          cudaOccupancyMaxActiveBlocksPerMultiprocessor(&fit, ks.persistent_ahead, block, bytes) == cudaSuccess &&
          (long long)fit * sms >= s->grid) break;
      cudaGetLastError();
    }
    s->n_stage = (int)ns; s->stage_smem = (size_t)ns * ks.stage_step_bytes;
    s->ahead = s->n_stage > 0 || s->prefetch;
    if (s->ahead) {      // the grid must be co-resident for this variant too
      int fit = 0;
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&fit, ks.persistent_ahead, block, s->stage_smem) != cudaSuccess ||
          (long long)fit * sms < s->grid) { cudaGetLastError(); s->ahead = false; s->n_stage = 0; s->stage_smem = 0; s->prefetch = 0; }
    }
  }
  // dedicated tail warps (k_persistent_dt) where the model's translation unit built them and nothing else was asked for:
  // default block size, no staged draws / prefetch chosen above, no TMA staging, no frozen-member hooks
  if (cfg->theta_mode == CUDAHM_THETA_DEVICE_TAIL && cfg->n_objects > 0 && ks.persistent_dt && !cfg->block_threads && !s->hold &&
      !s->ahead && !(cfg->flags & (CUDAHM_FLAG_TMA_STAGING | CUDAHM_FLAG_STAGE_STEPS_MASK | CUDAHM_FLAG_PREFETCH_ON))) {
    const long long per = (long long)s->vec * ks.dt_sweep_threads;
    s->dt = true;
    s->grid = (int)std::max(1LL, std::min<long long>(sms, (cfg->n_objects + per - 1) / per));
    s->block = ks.dt_sweep_threads + 128;
    s->sweep_grid = s->grid; s->sweep_block = ks.dt_sweep_threads;      // k_sweep at the same thread -> object map
    // own-thread staged draws: steps of plate draws made while the thread waits for the theta decision
    const long long steps = (cfg->n_objects + per * s->grid - 1) / (per * s->grid);
    long long ns = 2;                     // measured on C3: 0 -> 22.4, 1 -> 22.3, 2 -> 22.0, 3 -> 22.2, 4 -> 22.6 us per iteration
    ns = std::min<long long>(std::min(ns, steps), (long long)(STAGE_MAX_SMEM / (ks.stage_step_bytes * ks.dt_sweep_threads / block)));
    s->n_stage = (int)ns; s->stage_smem = (size_t)ns * (ks.stage_step_bytes * ks.dt_sweep_threads / block);
    // a handle that keeps no running moments runs the instantiation compiled without them (kernels.cuh, NO_MOM)
    if (!cfg->keep_chi_moments && ks.persistent_dt_nomom) s->ks.persistent_dt = ks.persistent_dt_nomom;
    if (ensure_dyn_smem(s->ks.persistent_dt, s->stage_smem) != cudaSuccess) { cudaGetLastError(); s->n_stage = 0; s->stage_smem = 0; }
  }
  // HBM-streaming variant with TMA-staged loads (stream_tma.cuh), opt-in: measured 10-30 % slower than plain vector
  // loads on C3 / C4 (the sweep is issue-bound, not latency-bound, and the producer warp costs a sweep warp)
  if (cfg->theta_mode == CUDAHM_THETA_DEVICE_TAIL && (cfg->flags & CUDAHM_FLAG_TMA_STAGING) && block <= 512 && ks.persistent_tma && !s->hold) {
    int stages = (int)std::min<size_t>(TMA_MAX_STAGES, (size_t)(200 * 1024) / ks.tma_stage_bytes);
    if (stages >= 2 && ensure_dyn_smem(ks.persistent_tma, stages * ks.tma_stage_bytes) == cudaSuccess) {
      s->tma_stages = stages; s->tma_smem = stages * ks.tma_stage_bytes;
      const long long tiles = (cfg->n_objects + (long long)s->vec * (block - 32) - 1) / ((long long)s->vec * (block - 32));
      s->grid = (int)std::max(1LL, std::min<long long>(sms, tiles));
    } else {
      cudaGetLastError();
    }
  }
  // on-chip variant: every object stays in the shared memory of its block for the whole launch
  if (cfg->theta_mode == CUDAHM_THETA_DEVICE_TAIL && !(cfg->flags & CUDAHM_FLAG_STREAMING_ONLY) && cfg->n_objects > 0 && !s->hold) {
    const int nv = rs.n_base + (cfg->keep_chi_moments ? 2 : 0);
    const void* rk = rs.kernel;
    if (rk) {
      const long long g = std::min<long long>(sms, (cfg->n_objects + 63) / 64);          // >= one warp of pairs per block
      const long long OB = 2 * ((cfg->n_objects + 2 * g - 1) / (2 * g));                   // objects per block (even)
      const long long R = 2 * ((OB + 2 * RES_S - 1) / (2 * RES_S));                        // slots per thread, in pairs
      const size_t bytes = (size_t)nv * R * RES_S * sizeof(double);
      if (R <= 2 && rs.kernel_sel_sweep) rk = rs.kernel_sel_sweep;      // short sweep: selection sum on the sweep warps
      if (bytes <= (size_t)RES_MAX_SMEM && ensure_dyn_smem(rk, bytes) == cudaSuccess) {
        s->res_kernel = rk; s->res_R = (int)R; s->res_OB = (int)OB; s->res_smem = bytes;
        s->grid = (int)g; s->block = RES_THREADS; s->res_threads = RES_THREADS; s->dt = false;
      } else {
        cudaGetLastError();
      }
    } else if (rs.gen_kernel) {
      // the general on-chip kernel: groups of `vec` adjacent objects per thread, 256 sweep threads per block; ONE object per
      // thread where that still covers the population (all sweep warps busy, half the serial work per thread)
      const bool one = rs.gen_kernel_v1 && cfg->n_objects <= (long long)sms * RG_S;
      const void* gk = one ? rs.gen_kernel_v1 : rs.gen_kernel;
      const long long vec = one ? 1 : rs.gen_vec;
      const long long g = std::min<long long>(sms, (cfg->n_objects + vec * 32 - 1) / (vec * 32));     // >= one warp of groups per block
      const long long OB = vec * ((cfg->n_objects + vec * g - 1) / (vec * g));                        // objects per block
      const long long R = vec * ((OB + vec * RG_S - 1) / (vec * RG_S));                               // slots per thread
      const size_t bytes = (size_t)rs.gen_values * R * RG_S * s->tsize;
      if (bytes <= (size_t)RES_MAX_SMEM && ensure_dyn_smem(gk, bytes) == cudaSuccess) {
        s->res_kernel = gk; s->res_R = (int)R; s->res_OB = (int)OB; s->res_smem = bytes;
        s->grid = (int)g; s->block = RG_THREADS; s->res_threads = RG_THREADS; s->dt = false;
      } else {
        cudaGetLastError();
      }
    }
  }

  Params& P = s->P;
  P.N = cfg->n_objects; P.Npad = (cfg->n_objects + 31) / 32 * 32;
  P.chi = s->ws + lay.chi; P.L = s->ws + lay.L; P.data = s->ws + lay.data;
  P.mom_mean = cfg->keep_chi_moments ? (double*)(s->ws + lay.mom_mean) : nullptr;
  P.mom_M2 = cfg->keep_chi_moments ? (double*)(s->ws + lay.mom_M2) : nullptr;
  P.slots = (double*)(s->ws + lay.slots); P.mbox = (unsigned long long*)(s->ws + lay.mbox);
  P.blk_cnt = (unsigned long long*)(s->ws + lay.blk_cnt);
  P.iter = (Iter*)(s->ws + lay.iter); P.trace = (double*)(s->ws + lay.trace); P.totals = (double*)(s->ws + lay.totals);
  P.qx = (double*)(s->ws + lay.qx); P.qex = (double*)(s->ws + lay.qex); P.qW = (double*)(s->ws + lay.qW);
  for (int k = 0; k < MC_N; ++k) P.mc[k] = 0.0;
  P.astar_chi = cfg->target_accept_chi;
  P.max_blocks = MAX_BLOCKS;
  P.tail = TailCfg{cfg->model, dt, cfg->freeze_theta ? 1 : 0, cfg->keep_chi_moments ? 1 : 0, cfg->seed,
                   cfg->target_accept_theta, cfg->eta_exponent, 0, cfg->max_trace_rows, 1, 0,
                   (double)(cfg->n_objects_total ? cfg->n_objects_total : cfg->n_objects), cfg->adapt_until, {}, {}};
  P.obj_offset = cfg->object_offset;
  P.rk = make_round_keys(cfg->seed);
  P.mask = cfg->update_mask ? (const unsigned char*)(s->ws + lay.mask) : nullptr;
  P.cnt = cfg->per_object_counter ? (unsigned*)(s->ws + lay.cnt) : nullptr;
  for (int j = 0; j < MAXD; ++j) { P.tail.prior_mean[j] = cfg->prior_mean[j]; P.tail.prior_isd[j] = cfg->prior_isd[j]; }
  P.taps = DevTaps{};

  if (cudaMemsetAsync(s->ws, 0, lay.total, s->stream) != cudaSuccess ||
      (cfg->update_mask && cudaMemsetAsync(s->ws + lay.mask, 1, (size_t)P.Npad, s->stream) != cudaSuccess) ||
      cudaHostAlloc((void**)&s->h_iter, sizeof(Iter), cudaHostAllocDefault) != cudaSuccess ||
      cudaHostAlloc((void**)&s->h_totals, NPART * sizeof(double), cudaHostAllocDefault) != cudaSuccess ||
      cudaEventCreate(&s->ev0) != cudaSuccess || cudaEventCreate(&s->ev1) != cudaSuccess) {
    const char* m = cudaGetErrorString(cudaGetLastError());
    cudahm_destroy(s);
    return fail(nullptr, CUDAHM_E_CUDA, "create: %s", m);
  }
  std::memset(s->h_iter, 0, sizeof(Iter));
  *out = s;
  return CUDAHM_OK;
}

extern "C" void cudahm_destroy(cudahm_sampler* s) {
  if (!s) return;
  cudaStreamSynchronize(s->stream);
  if (s->gexec) cudaGraphExecDestroy(s->gexec);
  drop_persistent_graph(s);
  if (s->h_iter) cudaFreeHost(s->h_iter);
  if (s->h_totals) cudaFreeHost(s->h_totals);
  if (s->ev0) cudaEventDestroy(s->ev0);
  if (s->ev1) cudaEventDestroy(s->ev1);
  delete s;
}

extern "C" int cudahm_sync(cudahm_sampler* s) {
  if (!s) return fail(nullptr, CUDAHM_E_INVALID, "NULL handle");
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  CU_TRY(s, cudaGetLastError());
  return CUDAHM_OK;
}

extern "C" int cudahm_set_data(cudahm_sampler* s, const void* const* cols, int n_cols, int cols_on_device) {
  if (!s || !cols) return fail(s, CUDAHM_E_INVALID, "set_data: NULL argument");
  if (n_cols != s->ncols) return fail(s, CUDAHM_E_INVALID, "set_data: model takes %d columns, got %d", s->ncols, n_cols);
  const long long N = s->P.N, Npad = s->P.Npad;
  const cudaMemcpyKind kind = cols_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  for (int c = 0; c < n_cols; ++c) {
    if (!cols[c] && N > 0) return fail(s, CUDAHM_E_INVALID, "set_data: column %d is NULL", c);
    if (N > 0) CU_TRY(s, cudaMemcpyAsync((char*)s->P.data + (size_t)c * Npad * s->tsize, cols[c], (size_t)N * s->tsize, kind, s->stream));
  }
  // Gaussian error columns sigma -> 1/(2 sigma^2)
  int first = -1, last = -1;
  switch (s->cfg.model) {
    case M_NORMAL1D: case M_LINREG_ME1D: first = last = 1; break;
    case M_BINORMAL2D: first = 2; last = 3; break;
    default: break;
  }
  if (N > 0) {
    const int tb = 256; const unsigned nb = (unsigned)((N + tb - 1) / tb);
    for (int c = first; c >= 0 && c <= last; ++c) {
      if (s->tsize == 8) k_sigma_to_h<double><<<nb, tb, 0, s->stream>>>((double*)s->P.data + (size_t)c * Npad, N);
      else k_sigma_to_h<float><<<nb, tb, 0, s->stream>>>((float*)s->P.data + (size_t)c * Npad, N);
      s->launches++;
    }
    CU_TRY(s, cudaGetLastError());
  }
  if (!cols_on_device) CU_TRY(s, cudaStreamSynchronize(s->stream));   // caller may free host buffers on return
  s->have_data = true; s->have_init = false;
  return CUDAHM_OK;
}

namespace {
// Gauss-Legendre rule on [a,b]: Newton on P_n from the Chebyshev-like guess; weights 2/((1-x^2) P_n'^2).
void gl_rule(int n, double a, double b, std::vector<double>& x, std::vector<double>& w) {
  x.assign(n, 0.0); w.assign(n, 0.0);
  const long double PI = 3.141592653589793238462643383279502884L;
  const long double half = 0.5L * ((long double)b - (long double)a), mid = 0.5L * ((long double)b + (long double)a);
  for (int i = 0; i < (n + 1) / 2; ++i) {
    long double t = cosl(PI * (4 * i + 3) / (4.0L * n + 2.0L)), d = 1.0L;
    for (int it = 0; it < 64; ++it) {
      long double pm = 1.0L, pc = t;
      for (int k = 1; k < n; ++k) { const long double pn = ((2 * k + 1) * t * pc - k * pm) / (k + 1); pm = pc; pc = pn; }
      d = n * (pm - t * pc) / (1.0L - t * t);
      const long double step = pc / d;
      t -= step;
      if (fabsl(step) < 1e-19L) {
        pm = 1.0L; pc = t;
        for (int k = 1; k < n; ++k) { const long double pn = ((2 * k + 1) * t * pc - k * pm) / (k + 1); pm = pc; pc = pn; }
        d = n * (pm - t * pc) / (1.0L - t * t);
        break;
      }
    }
    const long double wt = 2.0L / ((1.0L - t * t) * d * d);
    x[n - 1 - i] = (double)(mid + half * t); x[i] = (double)(mid - half * t);
    w[n - 1 - i] = w[i] = (double)(half * wt);
  }
}
}  // namespace

extern "C" int cudahm_set_model_consts(cudahm_sampler* s, const double* v, int n) {
  if (!s) return fail(s, CUDAHM_E_INVALID, "NULL handle");
  if (n != s->nconsts || (n > 0 && !v)) return fail(s, CUDAHM_E_INVALID, "model takes %d constants, got %d", s->nconsts, n);
  if (n == 0) { s->have_consts = true; return CUDAHM_OK; }
  if (normal_family_p(s->cfg.model) > 0) {
    // normal-normal family: {sigma_1..p, packed lower triangle of C_pop} (Eq. 3.3-3.4).  The kernels take
    // h_j = 1/(2 sigma_j^2) and Q = packed lower triangle of C_pop^-1 with the diagonal halved.  C_pop^-1 = G^-T G^-1 from
    // the Cholesky factor G of C_pop (long double; C_pop must be positive definite).
    const int np = normal_family_p(s->cfg.model);
    long double G[6][6] = {}, Gi[6][6] = {};
    const double* Cp = v + np;
    bool ok = true;
    for (int j = 0; j < np; ++j) ok = ok && v[j] > 0.0 && std::isfinite(v[j]);
    for (int r = 0; r < np && ok; ++r)
      for (int k = 0; k <= r; ++k) {
        long double a = Cp[r * (r + 1) / 2 + k];
        for (int m = 0; m < k; ++m) a -= G[r][m] * G[k][m];
        if (r == k) { ok = ok && a > 0.0L; G[r][r] = ok ? sqrtl(a) : 1.0L; }
        else G[r][k] = a / G[k][k];
      }
    if (!ok) return fail(s, CUDAHM_E_INVALID, "model constants out of range (sigma_j > 0, C_pop positive definite)");
    for (int c = 0; c < np; ++c)                       // Gi = G^-1 (lower triangular), column by column
      for (int r = c; r < np; ++r) {
        long double a = (r == c) ? 1.0L : 0.0L;
        for (int m = c; m < r; ++m) a -= G[r][m] * Gi[m][c];
        Gi[r][c] = a / G[r][r];
      }
    for (int j = 0; j < np; ++j) s->P.mc[MN_H + j] = 0.5 / (v[j] * v[j]);
    for (int r = 0; r < np; ++r)
      for (int c = 0; c <= r; ++c) {
        long double a = 0.0L;                          // (C^-1)_rc = sum_m Gi[m][r] Gi[m][c], m >= r
        for (int m = r; m < np; ++m) a += Gi[m][r] * Gi[m][c];
        s->P.mc[np + r * (r + 1) / 2 + c] = (double)(r == c ? 0.5L * a : a);
      }
    s->have_consts = true; s->have_init = false;
    invalidate_graph(s);
    return CUDAHM_OK;
  }
  std::vector<double> xk, wk, rj, wj, ex(NQUAD), W(NQUAD);
  if (s->cfg.model == M_THINNED_SCHECHTER1D) {
    // THINNED_SCHECHTER1D: {F_lim, sigma_F, x_lo, x_hi, r_min, r_max}
    if (!(v[MC_SIGF] > 0.0 && v[MC_XHI] > v[MC_XLO] && v[MC_RMAX] > v[MC_RMIN] && v[MC_RMIN] > 0.0))
      return fail(s, CUDAHM_E_INVALID, "model constants out of range");
    for (int k = 0; k < 6; ++k) s->P.mc[k] = v[k];
    s->P.mc[MC_INV2S2] = 0.5 / (v[MC_SIGF] * v[MC_SIGF]);
    // selection table: W_k = w_k * G(x_k), G(x) = int h(r) Phi((e^x/(4 pi r^2) - F_lim)/sigma_F) dr
    gl_rule(NQUAD, v[MC_XLO], v[MC_XHI], xk, wk);
    gl_rule(256, v[MC_RMIN], v[MC_RMAX], rj, wj);
    const double vol3 = (v[MC_RMAX] * v[MC_RMAX] * v[MC_RMAX] - v[MC_RMIN] * v[MC_RMIN] * v[MC_RMIN]) / 3.0;
    const double inv_s2 = 1.0 / (v[MC_SIGF] * std::sqrt(2.0));
    for (int k = 0; k < NQUAD; ++k) {
      ex[k] = std::exp(xk[k]);
      long double G = 0.0L;
      for (int j = 0; j < 256; ++j) {
        const double r2 = rj[j] * rj[j];
        const double F = ex[k] / (4.0 * M_PI * r2);
        G += (long double)(wj[j] * r2 * 0.5 * std::erfc((v[MC_FLIM] - F) * inv_s2));
      }
      W[k] = wk[k] * (double)(G / vol3);
    }
  } else {
    // BB1_FLUXNOISE1D: {sigma_0, alpha, x_lo, x_hi, r_min, r_max, F_th}.  eta(F) = Phi((F - F_th)/sigma(F)) with the
    // flux-dependent sigma of Eq. 5.8 does not depend on theta, so the 2-D cubature the paper
    // redoes for every proposal factorises here too: G(x) = int h(r) eta(e^x/(4 pi r^2)) dr is tabulated
    // once, by a 512-point rule in q = ln r (the detection edge has a fixed width in q wherever it falls).
    if (!(v[0] > 0.0 && v[1] >= 0.0 && v[MC_XHI] > v[MC_XLO] && v[MC_RMAX] > v[MC_RMIN] && v[MC_RMIN] > 0.0 && v[MB_FTH] > 0.0))
      return fail(s, CUDAHM_E_INVALID, "model constants out of range");
    for (int k = 0; k < 7; ++k) s->P.mc[k] = v[k];
    s->P.mc[MB_S0SQ] = v[0] * v[0]; s->P.mc[MB_A2] = v[1] * v[1];
    constexpr int NQR = 512;
    gl_rule(NQUAD, v[MC_XLO], v[MC_XHI], xk, wk);
    gl_rule(NQR, std::log(v[MC_RMIN]), std::log(v[MC_RMAX]), rj, wj);
    const double vol3 = (v[MC_RMAX] * v[MC_RMAX] * v[MC_RMAX] - v[MC_RMIN] * v[MC_RMIN] * v[MC_RMIN]) / 3.0;
    for (int k = 0; k < NQUAD; ++k) {
      ex[k] = std::exp(xk[k]);
      long double G = 0.0L;
      for (int j = 0; j < NQR; ++j) {
        const double F = ex[k] * std::exp(-2.0 * rj[j]) / (4.0 * M_PI);
        const double sg = std::sqrt(s->P.mc[MB_S0SQ] + s->P.mc[MB_A2] * F * F);
        G += (long double)(wj[j] * std::exp(3.0 * rj[j]) * 0.5 * std::erfc((v[MB_FTH] - F) / (sg * std::sqrt(2.0))));
      }
      W[k] = wk[k] * (double)(G / vol3);
    }
  }
  CU_TRY(s, cudaMemcpyAsync((void*)s->P.qx, xk.data(), NQUAD * 8, cudaMemcpyHostToDevice, s->stream));
  CU_TRY(s, cudaMemcpyAsync((void*)s->P.qex, ex.data(), NQUAD * 8, cudaMemcpyHostToDevice, s->stream));
  CU_TRY(s, cudaMemcpyAsync((void*)s->P.qW, W.data(), NQUAD * 8, cudaMemcpyHostToDevice, s->stream));
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  s->have_consts = true; s->have_init = false;
  invalidate_graph(s);
  return CUDAHM_OK;
}

// ----------------------------------------------------------------------------------------------------
namespace {

int launch(cudahm_sampler* s, const void* fn, int grid, int block, void** args, bool cooperative) {
  cudaError_t e = cooperative ? cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(block), args, 0, s->stream)
                              : cudaLaunchKernel(fn, dim3(grid), dim3(block), args, 0, s->stream);
  if (e != cudaSuccess) return fail(s, CUDAHM_E_CUDA, "kernel launch: %s", cudaGetErrorString(e));
  s->launches++;
  return CUDAHM_OK;
}

// upload a raw Iter (theta, L_theta, counters, t) and let the device derive the rest (k_init_iter)
int upload_and_init_iter(cudahm_sampler* s, const Iter& raw) {
  *s->h_iter = raw;
  CU_TRY(s, cudaMemcpyAsync(s->P.iter, s->h_iter, sizeof(Iter), cudaMemcpyHostToDevice, s->stream));
  Params P = s->P;
  void* args[] = {&P};
  int rc = launch(s, (const void*)k_init_iter, 1, 256, args, false);
  if (rc) return rc;
  CU_TRY(s, cudaMemcpyAsync(s->h_iter, s->P.iter, sizeof(Iter), cudaMemcpyDeviceToHost, s->stream));
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  s->host_iter_valid = true;
  // the chain must start where the theta target is positive and finite (X_1 with pi(X_1) > 0)
  if (!s->cfg.freeze_theta && (!std::isfinite(s->h_iter->lp_cur) || !std::isfinite(s->h_iter->T_cur)))
    return fail(s, CUDAHM_E_NONFINITE, "theta has zero prior density or a non-finite theta-only term (log prior %g, T %g)",
                s->h_iter->lp_cur, s->h_iter->T_cur);
  return CUDAHM_OK;
}

int fetch_iter(cudahm_sampler* s) {   // device -> h_iter (no-op in host mode, where h_iter is authoritative)
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  if (s->cfg.theta_mode == CUDAHM_THETA_HOST && s->host_iter_valid) return CUDAHM_OK;
  CU_TRY(s, cudaMemcpy(s->h_iter, s->P.iter, sizeof(Iter), cudaMemcpyDeviceToHost));
  return CUDAHM_OK;
}

}  // namespace

extern "C" int cudahm_set_init(cudahm_sampler* s, const void* chi0, int chi0_on_device, const double* theta0,
                               const double* theta_chol0) {
  if (!s || !theta0) return fail(s, CUDAHM_E_INVALID, "set_init: NULL argument");
  if (!s->have_data || !s->have_consts) return fail(s, CUDAHM_E_STATE, "set_init before set_data / set_model_consts");
  const long long N = s->P.N, Npad = s->P.Npad;
  if (chi0 && N > 0) {
    const cudaMemcpyKind kind = chi0_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    for (int j = 0; j < s->p; ++j)
      CU_TRY(s, cudaMemcpyAsync((char*)s->P.chi + (size_t)j * Npad * s->tsize, (const char*)chi0 + (size_t)j * N * s->tsize,
                                (size_t)N * s->tsize, kind, s->stream));
  }
  if (N > 0) {
    Params P = s->P;
    const void* raw = s->P.data;
    int have = chi0 ? 1 : 0;
    double sc64 = s->cfg.init_scale_chi; float sc32 = (float)sc64;
    void* args[] = {&P, &raw, &have, s->tsize == 8 ? (void*)&sc64 : (void*)&sc32};
    int rc = launch(s, s->ks.init_state, (int)((N + 255) / 256), 256, args, false);
    if (rc) return rc;
  }
  if (s->lay.trace != s->lay.totals)
    CU_TRY(s, cudaMemsetAsync(s->P.trace, 0, (size_t)s->cfg.max_trace_rows * s->dtheta * 8, s->stream));
  CU_TRY(s, cudaMemsetAsync(s->P.blk_cnt, 0, (size_t)MAX_BLOCKS * 2 * 8, s->stream));
  Iter raw;
  std::memset(&raw, 0, sizeof raw);
  for (int r = 0; r < s->dtheta; ++r) raw.theta[r] = theta0[r];
  if (theta_chol0) for (int k = 0; k < s->ntri_theta; ++k) raw.Lth[k] = theta_chol0[k];
  else for (int r = 0; r < s->dtheta; ++r) raw.Lth[tri(r, r)] = 0.1;
  raw.t = 1;
  s->t_done = 0; s->h_trace_rows = 0; s->h_mom_count = 0; s->h_proposals = 0;
  invalidate_graph(s);
  int rc = upload_and_init_iter(s, raw);
  if (rc) return rc;
  s->have_init = true;
  return CUDAHM_OK;
}

namespace {

// One cooperative launch of a persistent kernel, submitted as a one-node CUDA graph whose kernel parameters are updated in
// place: 2.3 us of host time per call (update 0.7 + launch 1.6) against 7.0 us for cudaLaunchCooperativeKernel, and on an
// idle stream the GPU waits for exactly that time.  The graph is kept as long as its executable:
// the in-place update names the NODE, which dies with the graph.  Falls back to the direct launch for good if any graph
// call fails; cudahm_stats.graph_launches tells which path a handle is on.
cudaError_t launch_persistent(cudahm_sampler* s, const void* fn, int grid, int block, void** args, size_t smem) {
  // the first launch of a handle goes out directly: building the graph costs ~100 us of host time, which a caller who runs
  // the whole chain in one cudahm_run should not pay before its kernel starts
  if (!s->pg_broken && s->pg_launches++ > 0) {
    cudaKernelNodeParams kp{};
    kp.func = const_cast<void*>(fn); kp.gridDim = dim3(grid); kp.blockDim = dim3(block); kp.sharedMemBytes = (unsigned)smem;
    kp.kernelParams = args; kp.extra = nullptr;
    cudaError_t e = cudaSuccess;
    if (!s->pg_exec || s->pg_fn != fn) {
      drop_persistent_graph(s);
      e = cudaGraphCreate(&s->pg_graph, 0);
      if (e == cudaSuccess) e = cudaGraphAddKernelNode(&s->pg_node, s->pg_graph, nullptr, 0, &kp);
      cudaKernelNodeAttrValue av{};
      av.cooperative = 1;
      if (e == cudaSuccess) e = cudaGraphKernelNodeSetAttribute(s->pg_node, cudaKernelNodeAttributeCooperative, &av);
      if (e == cudaSuccess) e = cudaGraphInstantiate(&s->pg_exec, s->pg_graph, 0);
      if (e == cudaSuccess) e = cudaGraphExecKernelNodeSetParams(s->pg_exec, s->pg_node, &kp);   // pays the lazy set-up of the update path now
      s->pg_fn = fn;
    } else {
      e = cudaGraphExecKernelNodeSetParams(s->pg_exec, s->pg_node, &kp);
    }
    if (e == cudaSuccess) e = cudaGraphLaunch(s->pg_exec, s->stream);
    if (e == cudaSuccess) { s->pg_graph_launches++; return e; }
    cudaGetLastError();
    drop_persistent_graph(s);
    s->pg_broken = true;
  }
  return cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(block), args, smem, s->stream);
}

// THETA_DEVICE_TAIL: cooperative persistent launches of at most max_it iterations each
int run_device_tail(cudahm_sampler* s, long long n_iter) {
  const long long max_it = 0x3fffffffLL;
  while (n_iter > 0) {
    long long k = std::min(n_iter, max_it);
    Params P = s->P;
    // mailbox epochs must never repeat while a stale slot could still hold them (0 = never written): before the 32-bit
    // counter would wrap, clear the mailboxes (stream-ordered) and start again at 1
    if ((unsigned long long)s->epoch + (unsigned long long)k >= 0xffffffffull) {
      CU_TRY(s, cudaMemsetAsync(s->ws + s->lay.mbox, 0, s->lay.blk_cnt - s->lay.mbox, s->stream));
      s->epoch = 1;
    }
    unsigned epoch0 = s->epoch;
    s->epoch += (unsigned)k;
    int R = s->res_R, OB = s->res_OB, ns = s->n_stage, pf = s->prefetch;
    void* args[] = {&P, &k, &epoch0, &R, &OB};
    void* pargs[] = {&P, &k, &epoch0, &ns, &pf};
    int rc;
    if (s->res_kernel) {
      cudaError_t e = ensure_dyn_smem(s->res_kernel, s->res_smem);      // a map lookup unless the limit has to grow
      if (e == cudaSuccess)
        e = launch_persistent(s, s->res_kernel, s->grid, s->res_threads, args, s->res_smem);
      if (e != cudaSuccess) return fail(s, CUDAHM_E_CUDA, "resident kernel launch: %s", cudaGetErrorString(e));
      s->launches++;
      rc = CUDAHM_OK;
    } else if (s->tma_stages > 0) {
      int st = s->tma_stages;
      void* targs[] = {&P, &k, &epoch0, &st};
      cudaError_t e = ensure_dyn_smem(s->ks.persistent_tma, s->tma_smem);
      if (e == cudaSuccess)
        e = launch_persistent(s, s->ks.persistent_tma, s->grid, s->block, targs, s->tma_smem);
      if (e != cudaSuccess) return fail(s, CUDAHM_E_CUDA, "streaming kernel launch: %s", cudaGetErrorString(e));
      s->launches++;
      rc = CUDAHM_OK;
    } else if (s->dt) {
      void* dargs[] = {&P, &k, &epoch0, &ns, &pf};
      cudaError_t e = launch_persistent(s, s->ks.persistent_dt, s->grid, s->block, dargs, s->stage_smem);
      if (e != cudaSuccess) return fail(s, CUDAHM_E_CUDA, "streaming kernel launch: %s", cudaGetErrorString(e));
      s->launches++;
      rc = CUDAHM_OK;
    } else {
      const void* fn = s->hold ? s->ks.persistent_hold : s->ahead ? s->ks.persistent_ahead : s->ks.persistent;
      cudaError_t e = s->ahead ? ensure_dyn_smem(fn, s->stage_smem) : cudaSuccess;
      if (e == cudaSuccess)
        e = launch_persistent(s, fn, s->grid, s->block, pargs, s->ahead ? s->stage_smem : 0);
      if (e != cudaSuccess) return fail(s, CUDAHM_E_CUDA, "persistent kernel launch: %s", cudaGetErrorString(e));
      s->launches++;
      rc = CUDAHM_OK;
    }
    if (rc) return rc;
    n_iter -= k;
  }
  return CUDAHM_OK;
}

int enqueue_graph_iteration(cudahm_sampler* s) {
  Params P = s->P;
  void* a1[] = {&P};
  int rc = launch(s, s->hold ? s->ks.sweep_hold : s->dt ? s->ks.sweep_dt : s->ks.sweep, s->sweep_grid, s->sweep_block, a1, false);
  if (rc) return rc;
  int nb = s->sweep_grid, flags = TAIL_DECIDE;
  void* a2[] = {&P, &nb, &flags};
  return launch(s, (const void*)k_tail, 1, TAIL_THREADS, a2, false);
}

// THETA_GRAPH: {sweep, tail} x GRAPH_ITERS captured once per (burn_in, thin), replayed; remainder launched directly
int run_graph(cudahm_sampler* s, long long n_iter) {
  constexpr int GRAPH_ITERS = 50;
  if (n_iter >= GRAPH_ITERS) {
    if (!s->gexec || s->g_burn != s->P.tail.burn_in || s->g_thin != s->P.tail.thin) {
      if (s->gexec) { cudaGraphExecDestroy(s->gexec); s->gexec = nullptr; }
      cudaStream_t cap;
      CU_TRY(s, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
      cudaStream_t user = s->stream;
      s->stream = cap;
      const long long before = s->launches;
      cudaGraph_t g = nullptr;
      cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
      int rc = CUDAHM_OK;
      if (e == cudaSuccess) {
        for (int k = 0; k < GRAPH_ITERS && rc == CUDAHM_OK; ++k) rc = enqueue_graph_iteration(s);
        e = cudaStreamEndCapture(cap, &g);
      }
      s->stream = user;
      s->launches = before;
      if (rc == CUDAHM_OK && e == cudaSuccess) e = cudaGraphInstantiate(&s->gexec, g, 0);
      if (g) cudaGraphDestroy(g);
      cudaStreamDestroy(cap);
      if (rc) return rc;
      if (e != cudaSuccess) return fail(s, CUDAHM_E_CUDA, "graph capture: %s", cudaGetErrorString(e));
      s->g_burn = s->P.tail.burn_in; s->g_thin = s->P.tail.thin; s->g_iters = GRAPH_ITERS;
    }
    while (n_iter >= GRAPH_ITERS) {
      CU_TRY(s, cudaGraphLaunch(s->gexec, s->stream));
      s->launches += 2 * GRAPH_ITERS;
      n_iter -= GRAPH_ITERS;
    }
  }
  for (; n_iter > 0; --n_iter) { int rc = enqueue_graph_iteration(s); if (rc) return rc; }
  return CUDAHM_OK;
}

// THETA_HOST (the paper's split): sweep + reduction on the device, theta step in host C++.
// Two halves, so that a sharded population can put its exchange between them (cudahm_shard_sweep / _decide).
int host_sweep(cudahm_sampler* s, void* totals_dev = nullptr) {   // -> s->h_totals = {S, Delta, Tq, n_accept, n_nonfinite} of this handle
  Params P = s->P;
  void* a1[] = {&P};
  int rc = launch(s, s->hold ? s->ks.sweep_hold : s->dt ? s->ks.sweep_dt : s->ks.sweep, s->sweep_grid, s->sweep_block, a1, false);
  if (rc) return rc;
  int nb = s->sweep_grid, flags = TAIL_REDUCE;
  void* a2[] = {&P, &nb, &flags};
  rc = launch(s, (const void*)k_tail, 1, TAIL_THREADS, a2, false);
  if (rc) return rc;
  if (totals_dev) {                            // the exchange runs on the device: leave the totals there, do not wait
    CU_TRY(s, cudaMemcpyAsync(totals_dev, s->P.totals, NPART * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
    return CUDAHM_OK;
  }
  CU_TRY(s, cudaMemcpyAsync(s->h_totals, s->P.totals, NPART * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  return CUDAHM_OK;
}
int host_decide(cudahm_sampler* s, const double* totals) {
  Iter& it = *s->h_iter;
  tail_decide(it, s->P.tail, totals);
  if (it.trace_write)
    CU_TRY(s, cudaMemcpyAsync(s->P.trace + (it.trace_rows - 1) * s->dtheta, it.theta, s->dtheta * sizeof(double),
                              cudaMemcpyHostToDevice, s->stream));
  prepare_iteration(it, s->P.tail, it.t + 1);
  CU_TRY(s, cudaMemcpyAsync(s->P.iter, s->h_iter, sizeof(Iter), cudaMemcpyHostToDevice, s->stream));
  // h_iter is pinned and reused next iteration: the copy must have left before we overwrite it
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  return CUDAHM_OK;
}
int run_host(cudahm_sampler* s, long long n_iter) {
  for (long long k = 0; k < n_iter; ++k) {
    int rc = host_sweep(s);
    if (!rc) rc = host_decide(s, s->h_totals);
    if (rc) return rc;
  }
  return CUDAHM_OK;
}

}  // namespace

extern "C" int cudahm_set_update_mask(cudahm_sampler* s, const uint8_t* mask, int mask_on_device) {
  if (!s) return fail(s, CUDAHM_E_INVALID, "NULL handle");
  if (!s->cfg.update_mask) return fail(s, CUDAHM_E_STATE, "set_update_mask needs cudahm_config.update_mask = 1");
  const size_t N = (size_t)s->P.N;
  unsigned char* dst = (unsigned char*)(s->ws + s->lay.mask);
  if (!mask) {
    CU_TRY(s, cudaMemsetAsync(dst, 1, (size_t)s->P.Npad, s->stream));
    s->n_active = (long long)N;
    return CUDAHM_OK;
  }
  std::vector<unsigned char> h(N);
  if (mask_on_device) {
    if (N) CU_TRY(s, cudaMemcpyAsync(dst, mask, N, cudaMemcpyDeviceToDevice, s->stream));
    if (N) CU_TRY(s, cudaMemcpyAsync(h.data(), mask, N, cudaMemcpyDeviceToHost, s->stream));
    CU_TRY(s, cudaStreamSynchronize(s->stream));
  } else {
    std::copy(mask, mask + N, h.begin());
    if (N) CU_TRY(s, cudaMemcpyAsync(dst, h.data(), N, cudaMemcpyHostToDevice, s->stream));
    CU_TRY(s, cudaStreamSynchronize(s->stream));      // h goes out of scope; the caller may free its buffer
  }
  long long k = 0;
  for (unsigned char m : h) k += m ? 1 : 0;
  s->n_active = k;
  return CUDAHM_OK;
}

extern "C" int cudahm_get_counters(cudahm_sampler* s, uint32_t* out) {
  if (!s || !out) return fail(s, CUDAHM_E_INVALID, "get_counters: NULL argument");
  if (!s->P.cnt) return fail(s, CUDAHM_E_STATE, "get_counters needs cudahm_config.per_object_counter = 1");
  if (!s->have_init) return fail(s, CUDAHM_E_STATE, "get_counters before set_init");
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  if (s->P.N) CU_TRY(s, cudaMemcpy(out, s->P.cnt, (size_t)s->P.N * 4, cudaMemcpyDeviceToHost));
  return CUDAHM_OK;
}

extern "C" int cudahm_set_counters(cudahm_sampler* s, const uint32_t* in) {
  if (!s || !in) return fail(s, CUDAHM_E_INVALID, "set_counters: NULL argument");
  if (!s->P.cnt) return fail(s, CUDAHM_E_STATE, "set_counters needs cudahm_config.per_object_counter = 1");
  if (!s->have_init) return fail(s, CUDAHM_E_STATE, "set_counters before set_init");
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  if (s->P.N) CU_TRY(s, cudaMemcpy(s->P.cnt, in, (size_t)s->P.N * 4, cudaMemcpyHostToDevice));
  return CUDAHM_OK;
}

extern "C" int cudahm_run(cudahm_sampler* s, int64_t n_iter, int64_t burn_in, int32_t thin) {
  if (!s) return fail(s, CUDAHM_E_INVALID, "NULL handle");
  if (!s->have_init) return fail(s, CUDAHM_E_STATE, "run before set_init");
  if (n_iter < 0 || burn_in < 0 || thin < 1) return fail(s, CUDAHM_E_INVALID, "run: bad n_iter/burn_in/thin");
  if (s->t_done + n_iter >= 0xffffffffLL) return fail(s, CUDAHM_E_INVALID, "iteration index exceeds the 32-bit stream counter");
  // trace capacity, from the host mirror of the row count: nothing is read back from the device (and the stream is not
  // synchronised) before the launch -- trace_rows and mom_count are functions of the (t, burn_in, thin) history alone
  const long long t1 = s->t_done + n_iter;
  const long long rows = s->cfg.max_trace_rows > 0 ? trace_rows_between(s->t_done, t1, burn_in, thin) : 0;
  if (s->cfg.max_trace_rows > 0 && s->h_trace_rows + rows > s->cfg.max_trace_rows)
    return fail(s, CUDAHM_E_INVALID, "theta trace would need %lld rows, capacity %lld", s->h_trace_rows + rows,
                (long long)s->cfg.max_trace_rows);
  s->P.tail.burn_in = burn_in; s->P.tail.thin = thin;
  if (n_iter == 0) return CUDAHM_OK;
  // the one call that may be made with any device current (a caller in a loop over handles need not switch): the handle's
  // device is made current for the duration of the call if it is not already
  struct DeviceScope {
    int prev = -1; bool switched = false;
    explicit DeviceScope(int want) { if (cudaGetDevice(&prev) == cudaSuccess && prev != want) switched = cudaSetDevice(want) == cudaSuccess; }
    ~DeviceScope() { if (switched) cudaSetDevice(prev); }
  } scope(s->device);
  const bool time_it = (s->cfg.flags & CUDAHM_FLAG_TIME_RUNS) != 0;
  if (time_it) CU_TRY(s, cudaEventRecord(s->ev0, s->stream));
  int rc;
  switch (s->cfg.theta_mode) {
    case CUDAHM_THETA_DEVICE_TAIL: rc = run_device_tail(s, n_iter); break;
    case CUDAHM_THETA_GRAPH:       rc = run_graph(s, n_iter); break;
    default:                       rc = run_host(s, n_iter); break;
  }
  if (rc) return rc;
  if (time_it) CU_TRY(s, cudaEventRecord(s->ev1, s->stream));
  s->timed = time_it;
  s->h_trace_rows += rows;
  if (s->cfg.keep_chi_moments) s->h_mom_count += moment_samples_between(s->t_done, t1, burn_in);
  s->h_proposals += n_iter * s->n_active;
  s->t_done = t1;
  return CUDAHM_OK;
}

// Sharded populations: the two halves of one THETA_HOST iteration, with the caller's exchange in between.
namespace {
int shard_check(cudahm_sampler* s, int64_t burn_in, int32_t thin, const void* p) {
  if (!s || !p) return fail(s, CUDAHM_E_INVALID, "shard: NULL argument");
  if (!s->have_init) return fail(s, CUDAHM_E_STATE, "shard call before set_init");
  if (s->cfg.theta_mode != CUDAHM_THETA_HOST) return fail(s, CUDAHM_E_UNSUPPORTED, "sharded stepping needs theta_mode = CUDAHM_THETA_HOST");
  if (burn_in < 0 || thin < 1) return fail(s, CUDAHM_E_INVALID, "shard: bad burn_in/thin");
  if (s->t_done + 1 >= 0xffffffffLL) return fail(s, CUDAHM_E_INVALID, "iteration index exceeds the 32-bit stream counter");
  s->P.tail.burn_in = burn_in; s->P.tail.thin = thin;
  return fetch_iter(s);
}
}  // namespace

extern "C" int cudahm_shard_sweep(cudahm_sampler* s, int64_t burn_in, int32_t thin, double* totals) {
  int rc = shard_check(s, burn_in, thin, totals);
  if (rc) return rc;
  rc = host_sweep(s);
  if (rc) return rc;
  for (int q = 0; q < NPART; ++q) totals[q] = s->h_totals[q];
  return CUDAHM_OK;
}

extern "C" int cudahm_shard_combine(const double* totals_by_rank, int n_ranks, double* out) {
  if (!totals_by_rank || !out || n_ranks < 1) return fail(nullptr, CUDAHM_E_INVALID, "shard_combine: bad argument");
  for (int q = 0; q < NPART; ++q) out[q] = totals_by_rank[q];
  for (int r = 1; r < n_ranks; ++r)                     // rank order; Tq (slot 2) is computed in full by every shard
    for (int q = 0; q < NPART; ++q)
      if (q != 2) out[q] += totals_by_rank[(size_t)r * NPART + q];
  return CUDAHM_OK;
}

extern "C" int cudahm_shard_sweep_device(cudahm_sampler* s, int64_t burn_in, int32_t thin, void* totals_dev) {
  int rc = shard_check(s, burn_in, thin, totals_dev);
  if (rc) return rc;
  return host_sweep(s, totals_dev);
}

extern "C" int cudahm_shard_decide(cudahm_sampler* s, int64_t burn_in, int32_t thin, const double* totals_global);
extern "C" int cudahm_shard_decide_gathered(cudahm_sampler* s, int64_t burn_in, int32_t thin, const void* gathered_dev,
                                            int n_ranks) {
  if (!s || !gathered_dev || n_ranks < 1 || n_ranks > 4096) return fail(s, CUDAHM_E_INVALID, "shard_decide_gathered: bad argument");
  std::vector<double> all((size_t)n_ranks * NPART);
  CU_TRY(s, cudaMemcpyAsync(all.data(), gathered_dev, all.size() * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  double tot[NPART];
  cudahm_shard_combine(all.data(), n_ranks, tot);
  return cudahm_shard_decide(s, burn_in, thin, tot);
}

extern "C" int cudahm_shard_decide(cudahm_sampler* s, int64_t burn_in, int32_t thin, const double* totals_global) {
  int rc = shard_check(s, burn_in, thin, totals_global);
  if (rc) return rc;
  const long long t = s->h_iter->t;
  if (s->cfg.max_trace_rows > 0 && t > burn_in && ((t - burn_in) % thin) == 0 && s->h_iter->trace_rows + 1 > s->cfg.max_trace_rows)
    return fail(s, CUDAHM_E_INVALID, "theta trace is full");
  rc = host_decide(s, totals_global);
  if (rc) return rc;
  s->t_done += 1;
  s->h_proposals += s->n_active;
  s->h_trace_rows = s->h_iter->trace_rows; s->h_mom_count = s->h_iter->mom_count;
  return CUDAHM_OK;
}

// ----------------------------------------------------------------------------------------------------
namespace {
// log C(beta, u, l), the BB1 normaliser of PAPER.md:429 (Eq. C.3): C = 1/(Gamma(b)(1 - (1 + u/l)^-b)), b = beta + 1 (both
// factors negative for b < 0); 1/log(1 + u/l) at b = 0.  Host only: the kernels work with rho/C (models.cuh).
double bb1_log_norm(const double* th) {
  const double b = th[0] + 1.0, A = std::log1p(std::exp(th[2] - th[1]));
  if (b == 0.0) return -std::log(A);
  return -(std::lgamma(b) + std::log(std::fabs(std::expm1(-b * A))));
}
}  // namespace

extern "C" int cudahm_debug_step(cudahm_sampler* s, int64_t burn_in, int32_t thin, cudahm_taps* taps) {
  if (!s || !taps) return fail(s, CUDAHM_E_INVALID, "debug_step: NULL argument");
  if (!s->have_init) return fail(s, CUDAHM_E_STATE, "debug_step before set_init");
  if (burn_in < 0 || thin < 1) return fail(s, CUDAHM_E_INVALID, "debug_step: bad burn_in/thin");
  int rc = fetch_iter(s); if (rc) return rc;
  if (s->cfg.theta_mode == CUDAHM_THETA_HOST)   // make the device copy current
    CU_TRY(s, cudaMemcpy(s->P.iter, s->h_iter, sizeof(Iter), cudaMemcpyHostToDevice));
  const long long t = s->h_iter->t;
  s->h_lp_prop_before = s->h_iter->lp_prop;
  if (s->cfg.max_trace_rows > 0 && t > burn_in && ((t - burn_in) % thin) == 0 &&
      s->h_iter->trace_rows + 1 > s->cfg.max_trace_rows)
    return fail(s, CUDAHM_E_INVALID, "theta trace is full");
  s->P.tail.burn_in = burn_in; s->P.tail.thin = thin;
  const size_t N = (size_t)s->P.N;
  // tap scratch is test instrumentation, not the hot path: allocated here, freed below
  const size_t nd = (size_t)(s->p + s->ntri + 6) * N;
  double* dbuf = nullptr; int* ibuf = nullptr;
  if (N > 0) {
    CU_TRY(s, cudaMalloc((void**)&dbuf, nd * sizeof(double)));
    if (cudaMalloc((void**)&ibuf, N * sizeof(int)) != cudaSuccess) { cudaFree(dbuf); return fail(s, CUDAHM_E_CUDA, "cudaMalloc taps"); }
  }
  Params P = s->P;
  double* q = dbuf;
  P.taps.chi_prop = q; q += (size_t)s->p * N;
  P.taps.L_new = q; q += (size_t)s->ntri * N;
  P.taps.pi_cur = q; q += N; P.taps.pi_prop = q; q += N; P.taps.alpha = q; q += N;
  P.taps.u = q; q += N; P.taps.a = q; q += N; P.taps.b = q; q += N;
  P.taps.accepted = ibuf;
  // constants the kernels drop (they cancel in every ratio): added back so the taps read in the paper's convention
  double lc = 0.0, lcp = 0.0;
  if (s->cfg.model == M_BB1_FLUXNOISE1D) { lc = bb1_log_norm(s->h_iter->theta); lcp = bb1_log_norm(s->h_iter->thetaP); }
  P.taps.shift_c = lc; P.taps.shift_p = lcp;
  const bool prop_in_support = s->h_iter->lp_prop != -INFINITY;
  void* a1[] = {&P};
  rc = launch(s, s->hold ? s->ks.sweep_tap_hold : s->dt ? s->ks.sweep_tap_dt : s->ks.sweep_tap, s->sweep_grid, s->sweep_block, a1, false);
  int nb = s->sweep_grid, flags = TAIL_REDUCE | TAIL_DECIDE;     // the device tail decides t and prepares t + 1
  void* a2[] = {&P, &nb, &flags};
  if (!rc) rc = launch(s, (const void*)k_tail, 1, TAIL_THREADS, a2, false);
  cudaError_t e = cudaSuccess;
  if (!rc) e = cudaMemcpyAsync(s->h_iter, s->P.iter, sizeof(Iter), cudaMemcpyDeviceToHost, s->stream);
  if (!rc && e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (!rc && e == cudaSuccess) {
    const Iter& it = *s->h_iter;
    for (int r = 0; r < 8; ++r) taps->theta_prop[r] = r < s->dtheta ? it.tap_thetaP[r] : 0.0;
    const double Nd = (double)s->P.N;
    taps->S = it.S + Nd * lc; taps->Delta = it.Delta + Nd * (lcp - lc);
    taps->T_cur = it.T_cur_used - Nd * lc; taps->T_prop = it.T_prop - (prop_in_support ? Nd * lcp : 0.0);
    taps->lp_cur = it.lp_cur_used; taps->lp_prop = s->h_lp_prop_before; taps->log_r = it.log_r;
    taps->alpha_theta = it.alpha_theta; taps->u_theta = it.u_theta; taps->accepted_theta = it.accepted_theta;
    struct { double* dst; const double* src; size_t n; } cp[] = {
        {taps->chi_prop, P.taps.chi_prop, (size_t)s->p * N}, {taps->L_new, P.taps.L_new, (size_t)s->ntri * N},
        {taps->pi_cur, P.taps.pi_cur, N}, {taps->pi_prop, P.taps.pi_prop, N}, {taps->alpha, P.taps.alpha, N},
        {taps->u, P.taps.u, N}, {taps->a, P.taps.a, N}, {taps->b, P.taps.b, N}};
    for (auto& c : cp)
      if (c.dst && c.n && e == cudaSuccess) e = cudaMemcpy(c.dst, c.src, c.n * sizeof(double), cudaMemcpyDeviceToHost);
    if (taps->accepted && N && e == cudaSuccess) e = cudaMemcpy(taps->accepted, ibuf, N * sizeof(int), cudaMemcpyDeviceToHost);
  }
  if (dbuf) cudaFree(dbuf);
  if (ibuf) cudaFree(ibuf);
  if (rc) return rc;
  if (e != cudaSuccess) return fail(s, CUDAHM_E_CUDA, "debug_step: %s", cudaGetErrorString(e));
  s->t_done += 1;
  s->h_proposals += s->n_active;
  s->h_trace_rows = s->h_iter->trace_rows; s->h_mom_count = s->h_iter->mom_count;
  return CUDAHM_OK;
}

// ----------------------------------------------------------------------------------------------------
// cudahm_debug_step_noalloc: the tapped iteration for callers that cannot call cudaMalloc (code under CUDA-graph capture,
// tight serving loops, harnesses that forbid it).  Same kernels, same launch shape, same taps as cudahm_debug_step; the tap
// scratch lives in ONE file-scope device array of CUDAHM_NOALLOC_SCRATCH_BYTES instead of a cudaMalloc per call.
//   - every GPU that loads the library holds the array until the process exits;
//   - in host code `g_noalloc_scratch` is a host-side STAND-IN for the symbol, not a device address: its device address is
//     looked up once per device, with that device current, by cudaGetSymbolAddress (noalloc_scratch_ptr) and only that
//     pointer is handed to the kernels;
//   - every call on a device shares the array, which keeps the previous call's contents: the range a call uses is cleared
//     (stream-ordered) before its kernels run, and calls that overlap on the GPU (two streams, two host threads) RACE.
namespace {
static __device__ __align__(256) unsigned char g_noalloc_scratch[CUDAHM_NOALLOC_SCRATCH_BYTES];

constexpr int NOALLOC_MAX_DEVICES = 64;
// device address of g_noalloc_scratch on the CURRENT device (resolved once per device); NULL + *err on failure
unsigned char* noalloc_scratch_ptr(cudaError_t* err) {
  static std::mutex mu;
  static unsigned char* ptr_of_device[NOALLOC_MAX_DEVICES] = {};
  int dev = -1;
  *err = cudaGetDevice(&dev);
  if (*err != cudaSuccess) return nullptr;
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) { *err = cudaErrorInvalidDevice; return nullptr; }
  std::lock_guard<std::mutex> lock(mu);
  if (!ptr_of_device[dev]) {
    void* q = nullptr;
    *err = cudaGetSymbolAddress(&q, g_noalloc_scratch);
    if (*err != cudaSuccess || !q) { if (*err == cudaSuccess) *err = cudaErrorInvalidSymbol; return nullptr; }
    ptr_of_device[dev] = static_cast<unsigned char*>(q);
  }
  return ptr_of_device[dev];
}
// bytes of tap scratch one tapped iteration of this handle needs: (p + ntri + 6) doubles and one int per object
size_t noalloc_bytes_needed(const cudahm_sampler* s) {
  const size_t N = (size_t)s->P.N;
  return align_up((size_t)(s->p + s->ntri + 6) * N * sizeof(double)) + N * sizeof(int);
}
}  // namespace

extern "C" size_t cudahm_debug_step_noalloc_bytes(const cudahm_sampler* s) { return s ? noalloc_bytes_needed(s) : 0; }

extern "C" int cudahm_debug_step_noalloc(cudahm_sampler* s, int64_t burn_in, int32_t thin, cudahm_taps* taps) {
  if (!s || !taps) return fail(s, CUDAHM_E_INVALID, "debug_step_noalloc: NULL argument");
  if (!s->have_init) return fail(s, CUDAHM_E_STATE, "debug_step_noalloc before set_init");
  if (burn_in < 0 || thin < 1) return fail(s, CUDAHM_E_INVALID, "debug_step_noalloc: bad burn_in/thin");
  const size_t N = (size_t)s->P.N;
  const size_t dbytes = align_up((size_t)(s->p + s->ntri + 6) * N * sizeof(double)), need = noalloc_bytes_needed(s);
  if (need > (size_t)CUDAHM_NOALLOC_SCRATCH_BYTES)      // refused before anything is touched: the handle stays usable
    return fail(s, CUDAHM_E_WORKSPACE,
                "debug_step_noalloc: %lld objects of this model need %zu bytes of tap scratch, the built-in array holds %zu "
                "(CUDAHM_NOALLOC_SCRATCH_BYTES); use cudahm_debug_step for larger populations",
                (long long)N, need, (size_t)CUDAHM_NOALLOC_SCRATCH_BYTES);
  cudaError_t e = cudaSuccess;
  unsigned char* const scratch = noalloc_scratch_ptr(&e);
  if (!scratch) return fail(s, CUDAHM_E_CUDA, "debug_step_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
  int rc = fetch_iter(s); if (rc) return rc;
  if (s->cfg.theta_mode == CUDAHM_THETA_HOST)   // make the device copy current
    CU_TRY(s, cudaMemcpy(s->P.iter, s->h_iter, sizeof(Iter), cudaMemcpyHostToDevice));
  const long long t = s->h_iter->t;
  s->h_lp_prop_before = s->h_iter->lp_prop;
  if (s->cfg.max_trace_rows > 0 && t > burn_in && ((t - burn_in) % thin) == 0 &&
      s->h_iter->trace_rows + 1 > s->cfg.max_trace_rows)
    return fail(s, CUDAHM_E_INVALID, "theta trace is full");
  s->P.tail.burn_in = burn_in; s->P.tail.thin = thin;
  // the array keeps the last call's taps (possibly another handle's): clear the range this call uses
  if (need > 0) CU_TRY(s, cudaMemsetAsync(scratch, 0, need, s->stream));
  double* const dbuf = reinterpret_cast<double*>(scratch);
  int* const ibuf = reinterpret_cast<int*>(scratch + dbytes);
  Params P = s->P;
  double* q = dbuf;
  P.taps.chi_prop = q; q += (size_t)s->p * N;
  P.taps.L_new = q; q += (size_t)s->ntri * N;
  P.taps.pi_cur = q; q += N; P.taps.pi_prop = q; q += N; P.taps.alpha = q; q += N;
  P.taps.u = q; q += N; P.taps.a = q; q += N; P.taps.b = q; q += N;
  P.taps.accepted = ibuf;
  double lc = 0.0, lcp = 0.0;
  if (s->cfg.model == M_BB1_FLUXNOISE1D) { lc = bb1_log_norm(s->h_iter->theta); lcp = bb1_log_norm(s->h_iter->thetaP); }
  P.taps.shift_c = lc; P.taps.shift_p = lcp;
  const bool prop_in_support = s->h_iter->lp_prop != -INFINITY;
  void* a1[] = {&P};
  rc = launch(s, s->hold ? s->ks.sweep_tap_hold : s->dt ? s->ks.sweep_tap_dt : s->ks.sweep_tap, s->sweep_grid, s->sweep_block, a1, false);
  int nb = s->sweep_grid, flags = TAIL_REDUCE | TAIL_DECIDE;
  void* a2[] = {&P, &nb, &flags};
  if (!rc) rc = launch(s, (const void*)k_tail, 1, TAIL_THREADS, a2, false);
  if (rc) return rc;
  e = cudaMemcpyAsync(s->h_iter, s->P.iter, sizeof(Iter), cudaMemcpyDeviceToHost, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e == cudaSuccess) {
    const Iter& it = *s->h_iter;
    for (int r = 0; r < 8; ++r) taps->theta_prop[r] = r < s->dtheta ? it.tap_thetaP[r] : 0.0;
    const double Nd = (double)s->P.N;
    taps->S = it.S + Nd * lc; taps->Delta = it.Delta + Nd * (lcp - lc);
    taps->T_cur = it.T_cur_used - Nd * lc; taps->T_prop = it.T_prop - (prop_in_support ? Nd * lcp : 0.0);
    taps->lp_cur = it.lp_cur_used; taps->lp_prop = s->h_lp_prop_before; taps->log_r = it.log_r;
    taps->alpha_theta = it.alpha_theta; taps->u_theta = it.u_theta; taps->accepted_theta = it.accepted_theta;
    struct { double* dst; const double* src; size_t n; } cp[] = {
        {taps->chi_prop, P.taps.chi_prop, (size_t)s->p * N}, {taps->L_new, P.taps.L_new, (size_t)s->ntri * N},
        {taps->pi_cur, P.taps.pi_cur, N}, {taps->pi_prop, P.taps.pi_prop, N}, {taps->alpha, P.taps.alpha, N},
        {taps->u, P.taps.u, N}, {taps->a, P.taps.a, N}, {taps->b, P.taps.b, N}};
    for (auto& c : cp)
      if (c.dst && c.n && e == cudaSuccess) e = cudaMemcpy(c.dst, c.src, c.n * sizeof(double), cudaMemcpyDeviceToHost);
    if (taps->accepted && N && e == cudaSuccess) e = cudaMemcpy(taps->accepted, ibuf, N * sizeof(int), cudaMemcpyDeviceToHost);
  }
  if (e != cudaSuccess) return fail(s, CUDAHM_E_CUDA, "debug_step_noalloc: %s", cudaGetErrorString(e));
  s->t_done += 1;
  s->h_proposals += s->n_active;
  s->h_trace_rows = s->h_iter->trace_rows; s->h_mom_count = s->h_iter->mom_count;
  return CUDAHM_OK;
}

extern "C" int cudahm_get_theta_trace(cudahm_sampler* s, double* out, int64_t cap_rows, int64_t* n_rows) {
  if (!s || !n_rows) return fail(s, CUDAHM_E_INVALID, "get_theta_trace: NULL argument");
  if (!s->have_init) return fail(s, CUDAHM_E_STATE, "get_theta_trace before set_init");
  // the count is mirrored on the host (a function of the (t, burn_in, thin) history): the query needs no synchronisation,
  // and the copy is ONE stream-ordered transfer followed by one synchronise -- no read-back of the iteration record first
  const long long rows = s->h_trace_rows;
  *n_rows = rows;
  if (!out) return CUDAHM_OK;
  if (cap_rows < rows) return fail(s, CUDAHM_E_INVALID, "trace has %lld rows, capacity %lld", rows, (long long)cap_rows);
  if (rows > 0) CU_TRY(s, cudaMemcpyAsync(out, s->P.trace, (size_t)rows * s->dtheta * 8, cudaMemcpyDeviceToHost, s->stream));
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  return CUDAHM_OK;
}

extern "C" int cudahm_get_chi_moments(cudahm_sampler* s, double* mean, double* var, int64_t cap_objects, int64_t* n_samples) {
  if (!s || !n_samples) return fail(s, CUDAHM_E_INVALID, "get_chi_moments: NULL argument");
  if (!s->have_init) return fail(s, CUDAHM_E_STATE, "get_chi_moments before set_init");
  if (!s->cfg.keep_chi_moments) return fail(s, CUDAHM_E_STATE, "keep_chi_moments was not set");
  // the sample count is mirrored on the host; the finalising kernel and every transfer are queued on the handle's stream
  // and synchronised ONCE (with pinned destinations the two arrays move back to back at PCIe speed)
  const long long cnt = s->h_mom_count, N = s->P.N, Npad = s->P.Npad;
  *n_samples = cnt;
  if (cap_objects < N) return fail(s, CUDAHM_E_INVALID, "moments need room for %lld objects", N);
  double* dvar = (double*)(s->ws + s->lay.mom_var);
  if (var && N > 0) {
    const long long n = (long long)s->p * Npad;
    const double inv = cnt > 1 ? 1.0 / (double)(cnt - 1) : 0.0;
    k_finalize_moments<<<(unsigned)((n + 255) / 256), 256, 0, s->stream>>>(s->P.mom_M2, dvar, n, inv);
    s->launches++;
    CU_TRY(s, cudaGetLastError());
  }
  for (int j = 0; j < s->p && N > 0; ++j)       // the means first: their transfer does not wait for the kernel's result
    if (mean) CU_TRY(s, cudaMemcpyAsync(mean + (size_t)j * N, s->P.mom_mean + (size_t)j * Npad, (size_t)N * 8, cudaMemcpyDeviceToHost, s->stream));
  for (int j = 0; j < s->p && N > 0; ++j)
    if (var) CU_TRY(s, cudaMemcpyAsync(var + (size_t)j * N, dvar + (size_t)j * Npad, (size_t)N * 8, cudaMemcpyDeviceToHost, s->stream));
  CU_TRY(s, cudaStreamSynchronize(s->stream));
  return CUDAHM_OK;
}

extern "C" int cudahm_get_stats(cudahm_sampler* s, cudahm_stats* out) {
  if (!s || !out) return fail(s, CUDAHM_E_INVALID, "get_stats: NULL argument");
  std::memset(out, 0, sizeof *out);
  out->grid_blocks = s->grid; out->block_threads = s->block; out->gpu_launches = s->launches;
  const bool streaming_tail = s->cfg.theta_mode == CUDAHM_THETA_DEVICE_TAIL && !s->res_kernel && s->tma_stages == 0 && (s->ahead || s->dt);
  out->dedicated_tail = (s->dt && !s->res_kernel) ? 1 : 0;
  out->graph_launches = s->pg_graph_launches;
  out->stage_steps = streaming_tail ? s->n_stage : 0; out->l2_prefetch = streaming_tail ? s->prefetch : 0;
  if (!s->have_init) return CUDAHM_OK;
  int rc = fetch_iter(s); if (rc) return rc;
  const Iter& it = *s->h_iter;
  out->iterations = it.t - 1;
  std::vector<unsigned long long> bc((size_t)2 * MAX_BLOCKS);
  CU_TRY(s, cudaMemcpy(bc.data(), s->P.blk_cnt, bc.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
  unsigned long long acc = it.chi_acc, nonf = it.nonfinite;
  for (int b = 0; b < MAX_BLOCKS; ++b) { acc += bc[2 * b]; nonf += bc[2 * b + 1]; }
  out->chi_accepts = (int64_t)acc; out->chi_proposals = s->h_proposals;   // iterations x updated objects of the WHOLE population (sharded: chi_acc is global too)
  out->theta_accepts = (int64_t)it.theta_acc; out->theta_proposals = (int64_t)it.theta_prop_n;
  out->nonfinite = (int64_t)nonf; out->moment_samples = it.mom_count; out->trace_rows = it.trace_rows;
  if (s->timed) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, s->ev0, s->ev1) == cudaSuccess) out->last_run_ms = ms;
  }
  return CUDAHM_OK;
}

extern "C" int cudahm_get_state(cudahm_sampler* s, void* chi, void* L, double* theta, double* L_theta, int64_t* t) {
  if (!s) return fail(s, CUDAHM_E_INVALID, "NULL handle");
  if (!s->have_init) return fail(s, CUDAHM_E_STATE, "get_state before set_init");
  int rc = fetch_iter(s); if (rc) return rc;
  const size_t N = (size_t)s->P.N, Npad = (size_t)s->P.Npad, ts = s->tsize;
  for (int j = 0; j < s->p && chi && N; ++j)
    CU_TRY(s, cudaMemcpy((char*)chi + j * N * ts, (char*)s->P.chi + j * Npad * ts, N * ts, cudaMemcpyDeviceToHost));
  for (int k = 0; k < s->ntri && L && N; ++k)
    CU_TRY(s, cudaMemcpy((char*)L + k * N * ts, (char*)s->P.L + k * Npad * ts, N * ts, cudaMemcpyDeviceToHost));
  if (theta) std::copy(s->h_iter->theta, s->h_iter->theta + s->dtheta, theta);
  if (L_theta) std::copy(s->h_iter->Lth, s->h_iter->Lth + s->ntri_theta, L_theta);
  if (t) *t = s->h_iter->t - 1;
  return CUDAHM_OK;
}

extern "C" int cudahm_set_state(cudahm_sampler* s, const void* chi, const void* L, const double* theta,
                                const double* L_theta, int64_t t) {
  if (!s || t < 0) return fail(s, CUDAHM_E_INVALID, "set_state: bad argument");
  if (!s->have_init) return fail(s, CUDAHM_E_STATE, "set_state before set_init");
  int rc = fetch_iter(s); if (rc) return rc;
  const size_t N = (size_t)s->P.N, Npad = (size_t)s->P.Npad, ts = s->tsize;
  for (int j = 0; j < s->p && chi && N; ++j)
    CU_TRY(s, cudaMemcpy((char*)s->P.chi + j * Npad * ts, (const char*)chi + j * N * ts, N * ts, cudaMemcpyHostToDevice));
  for (int k = 0; k < s->ntri && L && N; ++k)
    CU_TRY(s, cudaMemcpy((char*)s->P.L + k * Npad * ts, (const char*)L + k * N * ts, N * ts, cudaMemcpyHostToDevice));
  Iter raw = *s->h_iter;
  if (theta) std::copy(theta, theta + s->dtheta, raw.theta);
  if (L_theta) std::copy(L_theta, L_theta + s->ntri_theta, raw.Lth);
  raw.t = t + 1;
  s->t_done = t;
  s->h_proposals = t * (long long)s->P.tail.n_objects;
  if (s->P.cnt && N > 0) {       // as if every object had been updated in every iteration so far
    k_fill_u32<<<(unsigned)((N + 255) / 256), 256, 0, s->stream>>>(s->P.cnt, (long long)N, (unsigned)t);
    s->launches++;
    CU_TRY(s, cudaGetLastError());
  }
  invalidate_graph(s);
  return upload_and_init_iter(s, raw);
}
