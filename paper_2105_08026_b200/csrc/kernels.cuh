// kernels.cuh -- the fused plate sweep, its deterministic reduction, the grid barrier, the persistent
// Gibbs kernel and the small tail / setup kernels.  sm_100a.  DESIGN.md section 8.
//
// One sweep = RAM steps 1-3 for every object fused with the population terms
// a_i = log f(chi_i; theta), b_i = log f(chi_i; theta') that the theta step needs, the
// selection-integral slice and the running chi moments, in ONE pass over the SoA state.
#pragma once
#include <cuda_runtime.h>
#include "theta_step.cuh"

namespace hm {

struct DevTaps {
  double *chi_prop, *pi_cur, *pi_prop, *alpha, *u, *L_new, *a, *b;
  int* accepted;
};

struct Params {
  long long N, Npad;             // objects, column stride (multiple of 32)
  void* chi;                     // T [p][Npad]
  void* L;                       // T [ntri][Npad]
  void* data;                    // T [ncols][Npad], Gaussian error columns stored as 1/(2 sigma^2)
  double* mom_mean;              // [p][Npad]   Welford mean
  double* mom_M2;                // [p][Npad]   Welford sum of squared deviations
  double* slots;                 // [2][max_blocks][NPART] per-block partials, double-buffered by iteration parity
  unsigned* bar;                 // grid barrier arrival counter
  Iter* iter;                    // prepared iteration state (global copy)
  double* trace;                 // [max_trace_rows][dtheta]
  double* totals;                // [NPART] reduced totals (host mode reads them)
  const double* qx;              // [NQUAD] quadrature nodes x_k
  const double* qex;             // [NQUAD] e^{x_k}
  const double* qW;              // [NQUAD] W_k = w_k G(x_k)
  double mc[8];                  // model constants (MC_*)
  double astar_chi;
  int max_blocks, pad_;
  TailCfg tail;
  DevTaps taps;
};

template <class T> struct VecOf;
template <> struct VecOf<double> { using type = double2; static constexpr int n = 2; };
template <> struct VecOf<float>  { using type = float4;  static constexpr int n = 4; };

template <class T> __device__ __forceinline__ void ld_vec(const T* p, T* out, bool ro);
template <> __device__ __forceinline__ void ld_vec<double>(const double* p, double* out, bool ro) {
  const double2 v = ro ? __ldg(reinterpret_cast<const double2*>(p)) : *reinterpret_cast<const double2*>(p);
  out[0] = v.x; out[1] = v.y;
}
template <> __device__ __forceinline__ void ld_vec<float>(const float* p, float* out, bool ro) {
  const float4 v = ro ? __ldg(reinterpret_cast<const float4*>(p)) : *reinterpret_cast<const float4*>(p);
  out[0] = v.x; out[1] = v.y; out[2] = v.z; out[3] = v.w;
}
__device__ __forceinline__ void st_vec(double* p, const double* v) { *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]); }
__device__ __forceinline__ void st_vec(float* p, const float* v) { *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]); }

__device__ __forceinline__ double hm_sqrt(double x) { return sqrt(x); }
__device__ __forceinline__ float hm_sqrt(float x) { return sqrtf(x); }

// Draws of object i at iteration t.  fp64: draw 0 = accept uniform, draw 1 = Box-Muller pair.
// fp32: one call; x -> u1, y -> u2, z -> accept uniform.  Returns z = rad*(cs, sn) and the unit vector.
template <int P>
__device__ __forceinline__ void plate_draws(unsigned long long seed, long long i, uint32_t t, double* z, double* cs,
                                            double* sn, double* u) {
  const U4 r0 = stream(seed, KIND_PLATE, (uint64_t)i, t, 0u);
  *u = u01(r0.x, r0.y);
  const U4 r1 = stream(seed, KIND_PLATE, (uint64_t)i, t, 1u);
  const double u1 = u01(r1.x, r1.y), u2 = u01(r1.z, r1.w);
  const double rad = sqrt(-2.0 * log(u1));
  if (P == 1) { *cs = cospi(2.0 * u2); *sn = 0.0; z[0] = rad * *cs; }
  else { sincospi(2.0 * u2, sn, cs); z[0] = rad * *cs; z[1] = rad * *sn; }
}
template <int P>
__device__ __forceinline__ void plate_draws(unsigned long long seed, long long i, uint32_t t, float* z, float* cs,
                                            float* sn, float* u) {
  const U4 r = stream(seed, KIND_PLATE, (uint64_t)i, t, 0u);
  const float u1 = u01f(r.x), u2 = u01f(r.y);
  *u = u01f(r.z);
  const float rad = sqrtf(-2.0f * logf(u1));
  if (P == 1) { *cs = cospif(2.0f * u2); *sn = 0.0f; z[0] = rad * *cs; }
  else { sincospif(2.0f * u2, sn, cs); z[0] = rad * *cs; z[1] = rad * *sn; }
}

// ---------------------------------------------------------------------------------------------------
// The sweep.  Fixed thread -> object map: at step k the thread with global index gid owns the VEC
// consecutive objects starting at VEC*(k*nthreads + gid): unit-stride 16-byte loads/stores per column.
// part[NPART] receives this thread's partial sums in ascending object order.
template <int MODEL, class T, bool TAP>
__device__ __forceinline__ void sweep(const Params& P, const Iter& it, double* part) {
  constexpr int p = ModelDims<MODEL>::p, ntri = p * (p + 1) / 2, ncols = ModelDims<MODEL>::ncols;
  constexpr int VEC = VecOf<T>::n;
  const long long N = P.N, Npad = P.Npad;
  const long long nthreads = (long long)gridDim.x * blockDim.x;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  T* const chi = static_cast<T*>(P.chi);
  T* const Lm = static_cast<T*>(P.L);
  const T* const dat = static_cast<const T*>(P.data);

  const uint32_t t = (uint32_t)it.t;
  const ThetaK kc = it.kc, kp = it.kp;
  const KT<T> kT = narrow<T>(kc);
  T mcT[7];
#pragma unroll
  for (int j = 0; j < 7; ++j) mcT[j] = (T)P.mc[j];
  const T eta = (T)it.eta, astar = (T)P.astar_chi;
  const bool do_mom = P.tail.keep_moments && it.t > P.tail.burn_in;
  const double inv_k = 1.0 / (double)(it.mom_count + 1);

  double accS = 0.0, accD = 0.0, nacc = 0.0, nnan = 0.0;

  for (long long base = (long long)VEC * gid; base < N; base += (long long)VEC * nthreads) {
    T x[p][VEC], l[ntri][VEC], d[ncols][VEC];
#pragma unroll
    for (int j = 0; j < p; ++j) ld_vec<T>(chi + j * Npad + base, x[j], false);
#pragma unroll
    for (int k = 0; k < ntri; ++k) ld_vec<T>(Lm + k * Npad + base, l[k], false);
#pragma unroll
    for (int c = 0; c < ncols; ++c) ld_vec<T>(dat + c * Npad + base, d[c], true);

#pragma unroll
    for (int v = 0; v < VEC; ++v) {
      const long long i = base + v;
      const bool live = i < N;
      T xi[p], di[ncols], z[2] = {T(0), T(0)}, cs, sn, u;
#pragma unroll
      for (int j = 0; j < p; ++j) xi[j] = x[j][v];
#pragma unroll
      for (int c = 0; c < ncols; ++c) di[c] = d[c][v];
      plate_draws<p>(P.tail.seed, i, t, z, &cs, &sn, &u);
      // step 1: chi' = chi + L z
      T yi[p];
      yi[0] = xi[0] + l[0][v] * z[0];
      if (p == 2) yi[1] = xi[1] + l[1][v] * z[0] + l[2][v] * z[1];
      // step 2: alpha = min{1, pi(chi')/pi(chi)}
      using PL = Plate<MODEL, T>;
      const typename PL::Pt qc = PL::point(xi), qp = PL::point(yi);
      const T pc = PL::target(qc, di, kT, mcT), pp = PL::target(qp, di, kT, mcT);
      const T diff = pp - pc;
      const bool bad = diff != diff;
      const T la = bad ? T(-INFINITY) : (diff < T(0) ? diff : T(0));
      const T alpha = hm_exp(la);
      const bool acc = u < alpha;
      const typename PL::Pt qn = acc ? qp : qc;
#pragma unroll
      for (int j = 0; j < p; ++j) x[j][v] = acc ? yi[j] : xi[j];
      // step 3: L <- L chol(I + c uu^T), u = z/|z| = (cs, sn)
      const T c = eta * (alpha - astar);
      T ln[ntri];
      if (p == 1) {
        ln[0] = l[0][v] * hm_sqrt(T(1) + c);
      } else {
        const T s1 = T(1) + c * cs * cs;
        const T k00 = hm_sqrt(s1);
        const T k10 = c * cs * sn / k00;
        const T k11 = hm_sqrt((T(1) + c) / s1);
        ln[0] = l[0][v] * k00;
        ln[1] = l[1][v] * k00 + l[2][v] * k10;
        ln[2] = l[2][v] * k11;
      }
      // population terms at the new chi, fp64
      const double a = PL::pop(qn, di, kc), b = PL::pop(qn, di, kp);
      if (live) {
#pragma unroll
        for (int k = 0; k < ntri; ++k) l[k][v] = ln[k];
        accS += a; accD += b - a;
        nacc += acc ? 1.0 : 0.0; nnan += bad ? 1.0 : 0.0;
        if (do_mom) {
#pragma unroll
          for (int j = 0; j < p; ++j) {
            const long long q = j * Npad + i;
            const double xv = (double)x[j][v];
            const double m0 = P.mom_mean[q];
            const double dl = xv - m0;
            const double m1 = m0 + dl * inv_k;
            P.mom_mean[q] = m1;
            P.mom_M2[q] += dl * (xv - m1);
          }
        }
        if (TAP) {
          const DevTaps& tp = P.taps;
#pragma unroll
          for (int j = 0; j < p; ++j) if (tp.chi_prop) tp.chi_prop[j * N + i] = (double)yi[j];
          if (tp.pi_cur) tp.pi_cur[i] = (double)pc;
          if (tp.pi_prop) tp.pi_prop[i] = (double)pp;
          if (tp.alpha) tp.alpha[i] = (double)alpha;
          if (tp.u) tp.u[i] = (double)u;
          if (tp.accepted) tp.accepted[i] = acc ? 1 : 0;
#pragma unroll
          for (int k = 0; k < ntri; ++k) if (tp.L_new) tp.L_new[k * N + i] = (double)ln[k];
          if (tp.a) tp.a[i] = a;
          if (tp.b) tp.b[i] = b;
        }
      } else {
#pragma unroll
        for (int j = 0; j < p; ++j) x[j][v] = xi[j];
      }
    }
#pragma unroll
    for (int j = 0; j < p; ++j) st_vec(chi + j * Npad + base, x[j]);
#pragma unroll
    for (int k = 0; k < ntri; ++k) st_vec(Lm + k * Npad + base, l[k]);
  }

  // selection-integral slice (M1): term k belongs to block k % gridDim.x, thread k / gridDim.x
  double tq = 0.0;
  if (MODEL == M_THINNED_SCHECHTER1D && !P.tail.freeze_theta) {
    for (int k = (int)blockIdx.x + (int)gridDim.x * (int)threadIdx.x; k < NQUAD; k += (int)gridDim.x * (int)blockDim.x)
      tq += P.qW[k] * exp(kp.v[0] * (P.qx[k] - kp.v[1]) - P.qex[k] * kp.v[3]);
  }
  part[0] = accS; part[1] = accD; part[2] = tq; part[3] = nacc; part[4] = nnan;
}

// Deterministic block reduction: shuffle tree inside each warp, then warp 0 over the per-warp results.
// Returns the block totals in part[] of thread 0.  red: shared [32][NPART].
__device__ __forceinline__ void block_reduce(double* part, double (*red)[NPART]) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int q = 0; q < NPART; ++q) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part[q] += __shfl_down_sync(0xffffffffu, part[q], o);
  }
  if (lane == 0) {
#pragma unroll
    for (int q = 0; q < NPART; ++q) red[wid][q] = part[q];
  }
  __syncthreads();
  if (wid == 0) {
#pragma unroll
    for (int q = 0; q < NPART; ++q) {
      double v = lane < nw ? red[lane][q] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
      part[q] = v;
    }
  }
}

// Fixed-order sum of the per-block slots by warp 0: lane l adds blocks l, l+32, ... in order, then a tree.
__device__ __forceinline__ void slots_reduce(const double* slots, int nblocks, double* tot) {
  const int lane = threadIdx.x & 31;
  double v[NPART];
#pragma unroll
  for (int q = 0; q < NPART; ++q) v[q] = 0.0;
  for (int g = lane; g < nblocks; g += 32) {
#pragma unroll
    for (int q = 0; q < NPART; ++q) v[q] += __ldcg(slots + (size_t)g * NPART + q);
  }
#pragma unroll
  for (int q = 0; q < NPART; ++q) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_down_sync(0xffffffffu, v[q], o);
    tot[q] = v[q];
  }
}

// Grid barrier for the co-resident (cooperative) grid: one release-add per block, one acquire-poll.
__device__ __forceinline__ void grid_barrier(unsigned* bar, unsigned target) {
  if (threadIdx.x == 0) {
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
    unsigned v;
    do {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
    } while (v < target);
  }
  __syncthreads();
}

__device__ __forceinline__ void copy_iter(Iter* dst, const Iter* src) {
  const int n = (int)(sizeof(Iter) / sizeof(double));
  const double* s = reinterpret_cast<const double*>(src);
  double* d = reinterpret_cast<double*>(dst);
  for (int k = threadIdx.x; k < n; k += blockDim.x) d[k] = s[k];
}
static_assert(sizeof(Iter) % sizeof(double) == 0, "Iter is copied as doubles");

// ---------------------------------------------------------------------------------------------------
// THETA_DEVICE_TAIL: the whole Gibbs loop in one cooperative launch.  Per iteration: sweep -> per-block
// slot -> ONE grid barrier -> every block reduces all slots in the same fixed order and thread 0 takes the
// identical theta decision (no second barrier; slots are double-buffered by iteration parity so a fast
// block's iteration t+1 write cannot race a slow block's iteration t read).
template <int MODEL, class T, int BLOCK>
__global__ void __launch_bounds__(BLOCK, 1) k_persistent(const Params P, const long long n_iter) {
  __shared__ Iter it;
  __shared__ double red[32][NPART];
  copy_iter(&it, P.iter);
  __syncthreads();
  const int G = (int)gridDim.x;
  for (long long k = 0; k < n_iter; ++k) {
    double part[NPART];
    sweep<MODEL, T, false>(P, it, part);
    block_reduce(part, red);
    double* slots = P.slots + (size_t)(k & 1) * P.max_blocks * NPART;
    if (threadIdx.x == 0) {
#pragma unroll
      for (int q = 0; q < NPART; ++q) __stcg(slots + (size_t)blockIdx.x * NPART + q, part[q]);
    }
    grid_barrier(P.bar, (unsigned)(k + 1) * (unsigned)G);
    if (threadIdx.x < 32) {
      double tot[NPART];
      slots_reduce(slots, G, tot);
      if (threadIdx.x == 0) {
        tail_decide(it, P.tail, tot);
        if (blockIdx.x == 0 && it.trace_write) {
          for (int j = 0; j < P.tail.dtheta; ++j) P.trace[(it.trace_rows - 1) * P.tail.dtheta + j] = it.theta[j];
        }
        prepare_iteration(it, P.tail, it.t + 1);
      }
    }
    __syncthreads();
  }
  if (blockIdx.x == 0) copy_iter(P.iter, &it);
}

// One sweep as its own launch (THETA_GRAPH, THETA_HOST, debug_step).  Same grid, same maps, same order.
template <int MODEL, class T, int BLOCK, bool TAP>
__global__ void __launch_bounds__(BLOCK, 1) k_sweep(const Params P) {
  __shared__ Iter it;
  __shared__ double red[32][NPART];
  copy_iter(&it, P.iter);
  __syncthreads();
  double part[NPART];
  sweep<MODEL, T, TAP>(P, it, part);
  block_reduce(part, red);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < NPART; ++q) P.slots[(size_t)blockIdx.x * NPART + q] = part[q];
  }
}

// 1-warp tail: reduce the slots; optionally decide; optionally prepare the next iteration.
enum : int { TAIL_REDUCE = 1, TAIL_DECIDE = 2, TAIL_PREPARE = 4 };
__global__ void __launch_bounds__(32, 1) k_tail(const Params P, const int nblocks, const int flags) {
  __shared__ Iter it;
  copy_iter(&it, P.iter);
  __syncwarp();
  double tot[NPART];
  if (flags & TAIL_REDUCE) {
    slots_reduce(P.slots, nblocks, tot);
    if (threadIdx.x == 0) {
#pragma unroll
      for (int q = 0; q < NPART; ++q) P.totals[q] = tot[q];
    }
  }
  if (threadIdx.x == 0) {
    if (flags & TAIL_DECIDE) {
      tail_decide(it, P.tail, tot);
      if (it.trace_write) {
        for (int j = 0; j < P.tail.dtheta; ++j) P.trace[(it.trace_rows - 1) * P.tail.dtheta + j] = it.theta[j];
      }
    }
    if (flags & TAIL_PREPARE) prepare_iteration(it, P.tail, (flags & TAIL_DECIDE) ? it.t + 1 : it.t);
  }
  __syncwarp();
  if (flags & (TAIL_DECIDE | TAIL_PREPARE)) copy_iter(P.iter, &it);
}

// After set_init / set_state: derive kc, log prior and T(theta) for the uploaded theta, then prepare it.t.
__global__ void __launch_bounds__(256, 1) k_init_iter(const Params P) {
  __shared__ Iter it;
  __shared__ double red[32][NPART];
  copy_iter(&it, P.iter);
  __syncthreads();
  const ThetaK kc = theta_consts(P.tail.model, it.theta);
  double part[NPART] = {0, 0, 0, 0, 0};
  if (P.tail.model == M_THINNED_SCHECHTER1D) {
    for (int k = threadIdx.x; k < NQUAD; k += blockDim.x)
      part[2] += P.qW[k] * exp(kc.v[0] * (P.qx[k] - kc.v[1]) - P.qex[k] * kc.v[3]);
  }
  block_reduce(part, red);
  if (threadIdx.x == 0) {
    it.kc = kc;
    it.lp_cur = log_prior(P.tail.model, it.theta);
    it.T_cur = (P.tail.model == M_THINNED_SCHECHTER1D) ? -exp(kc.v[2]) * part[2] : 0.0;
    prepare_iteration(it, P.tail, it.t);
  }
  __syncthreads();
  copy_iter(P.iter, &it);
}

// ---------------------------------------------------------------------------------------------------
// set-up kernels
// Gaussian error columns sigma -> h = 1/(2 sigma^2) (done once; removes every division from the sweep)
template <class T>
__global__ void k_sigma_to_h(T* col, long long N) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < N) { const T s = col[i]; col[i] = T(0.5) / (s * s); }
}

// default X_1 (pi(X_1) > 0) from the RAW data columns, L = scale * I, moments cleared
template <int MODEL, class T>
__global__ void k_init_state(const Params P, const T* raw, const int have_chi0, const T scale) {
  constexpr int p = ModelDims<MODEL>::p, ntri = p * (p + 1) / 2;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P.N) return;
  T* chi = static_cast<T*>(P.chi);
  T* Lm = static_cast<T*>(P.L);
  if (!have_chi0) {
    if (MODEL == M_THINNED_SCHECHTER1D) {
      double x = log((double)raw[i] / (double)raw[P.Npad + i]);
      x = fmin(fmax(x, P.mc[MC_XLO]), P.mc[MC_XHI]);
      chi[i] = (T)x;
    } else {
#pragma unroll
      for (int j = 0; j < p; ++j) chi[j * P.Npad + i] = raw[j * P.Npad + i];
    }
  }
#pragma unroll
  for (int k = 0; k < ntri; ++k) Lm[k * P.Npad + i] = T(0);
#pragma unroll
  for (int r = 0; r < p; ++r) Lm[(r * (r + 1) / 2 + r) * P.Npad + i] = scale;
  if (P.mom_mean) {
#pragma unroll
    for (int j = 0; j < p; ++j) { P.mom_mean[j * P.Npad + i] = 0.0; P.mom_M2[j * P.Npad + i] = 0.0; }
  }
}

// sample variance from the Welford sums, written next to them for read-out
__global__ void k_finalize_moments(const double* M2, double* var, long long n, double inv_km1) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) var[i] = M2[i] * inv_km1;
}

}  // namespace hm
