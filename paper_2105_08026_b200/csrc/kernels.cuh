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
  // additive constants the kernels drop because they cancel in every ratio (M4: log C(theta), log C(theta')); the taps
  // add them back so that they read in the paper's convention
  double shift_c, shift_p;
};

struct Params {
  long long N, Npad;             // objects, column stride (multiple of 32)
  void* chi;                     // T [p][Npad]
  void* L;                       // T [ntri][Npad]
  void* data;                    // T [ncols][Npad], Gaussian error columns stored as 1/(2 sigma^2)
  double* mom_mean;              // [p][Npad]   Welford mean
  double* mom_M2;                // [p][Npad]   Welford sum of squared deviations
  double* slots;                 // [max_blocks][NPART] per-block partials of k_sweep (THETA_GRAPH / HOST / debug_step)
  unsigned long long* mbox;      // [2][G][2][G][2] flagged mailboxes of k_persistent (G = its grid <= MAX_PGRID)
  unsigned long long* blk_cnt;   // [max_blocks][2] accepted / non-finite plate proposals counted by k_persistent
  Iter* iter;                    // prepared iteration state (global copy)
  double* trace;                 // [max_trace_rows][dtheta]
  double* totals;                // [NPART] reduced totals (host mode reads them)
  const double* qx;              // [NQUAD] quadrature nodes x_k
  const double* qex;             // [NQUAD] e^{x_k}
  const double* qW;              // [NQUAD] W_k = w_k G(x_k)
  double mc[MC_N];               // model constants (MC_* / MB_* / MN_*)
  double astar_chi;
  int max_blocks, pad_;
  long long obj_offset;          // global index of object 0 (sharded populations; even): keys the plate Philox streams
  // frozen members, read by the HOLD kernel variants only
  const unsigned char* mask;     // [Npad] 1 = update object i, 0 = hold it fixed; NULL = update everything
  unsigned* cnt;                 // [Npad] RAM updates object i has taken (eta_n from the object's own count); NULL = global n
  TailCfg tail;
  DevTaps taps;
  RoundKeys rk;                  // Philox round keys of tail.seed (philox.cuh)
};

// named barriers of the kernels with dedicated tail warps (resident.cuh, resident_gen.cuh, k_persistent_dt)
__device__ __forceinline__ void bar_sync(const int id, const int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive(const int id, const int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
enum : int { BAR_PARTIALS = 1, BAR_THETA = 2, BAR_TAIL = 3, BAR_THETAP = 4 };

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
// sqrt of a positive normal number as x * rsqrt(x) (<= 2 ulp): the RAM scale factor sqrt(1 + c), 1 + c in (0.4, 2)
__device__ __forceinline__ double hm_rsqrt(double x) { return rsqrt(x); }
// fp32: the hardware reciprocal square root on a NORMAL positive argument.  rsqrtf() wraps the same MUFU.RSQ in a subnormal
// pre-scale and post-scale (a compare and two multiplies, issued predicated off on every call); every argument here is
// normal -- -2 ln u1 >= 1.19e-7 for u1 <= 1 - 2^-24, 1 + c >= 1 - alpha*, |z|^2 and s_j s_j+1 of such terms -- so the .ftz
// form returns the same bits without them (a subnormal argument would flush to zero and return +inf).
__device__ __forceinline__ float hm_rsqrt(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ double hm_sqrt_pos(double x) { return hm_sqrt_fast(x); }
__device__ __forceinline__ void hm_sqrt_both(double x, double* g, double* ig) { hm_sqrt_rsqrt(x, g, ig); }
__device__ __forceinline__ void hm_sqrt_both(float x, float* g, float* ig) { *ig = hm_rsqrt(x); *g = x * *ig; }
__device__ __forceinline__ float hm_sqrt_pos(float x) { return x * hm_rsqrt(x); }

// Plate-level draws.  Objects draw in PAIRS m = i >> 1 so that one Philox call and one
// Box-Muller evaluation serve two objects (both Box-Muller branches are independent N(0,1); nothing is wasted):
//   fp64  p = 1: ONE call per pair (draw 0 of pair m), every word a 32-bit uniform (w + 1/2) 2^-32: x -> u1, y -> u2, cos /
//                sin branch, accept uniforms z / w.  (Half the Philox work of 52-bit uniforms; the proposal stays symmetric.)
//         p >= 2: accept uniforms (52 bits): draw 0 of pair m -- (x,y) for the even object, (z,w) for the odd one;
//                normals: per object, draw 1 of object i; z = rad*(cs, sn), unit vector (cs, sn).
//   fp32  p = 1: one call per pair (draw 0 of pair m): x -> u1, y -> u2, cos / sin branch, accept uniforms z / w.
// i0 is the even object of the pair.  z[h][k]: normal k of object i0 + h.
//         p >= 3 normals:  per object, draws 1 + k of object i give (z_2k, z_2k+1), k = 0 .. ceil(p/2) - 1.
template <int P, int ZD, class KEY>
__device__ __forceinline__ void pair_draws(const KEY& seed, long long i0, uint32_t t, double (*z)[ZD], double* cs,
                                           double* sn, double* u) {
  const uint64_t m = (uint64_t)i0 >> 1;
  const U4 a = stream(seed, KIND_PLATE, m, t, 0u);
  if (P == 1) {
    const double u1 = u01_32(a.x), u2 = u01_32(a.y);
    u[0] = u01_32(a.z); u[1] = u01_32(a.w);
    const double rad = hm_sqrt_fast(-2.0 * hm_log_unit(u1));
    double s_, c_;
    hm_sincos2pi(u2, &s_, &c_);
    z[0][0] = rad * c_; z[1][0] = rad * s_;
    z[0][1] = 0.0; z[1][1] = 0.0;
    cs[0] = cs[1] = 0.0; sn[0] = sn[1] = 0.0;      // the unit vector is not needed for p = 1
  } else {
    u[0] = u01(a.x, a.y); u[1] = u01(a.z, a.w);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const U4 b = stream(seed, KIND_PLATE, (uint64_t)(i0 + h), t, 1u);
      const double u1 = u01(b.x, b.y), u2 = u01(b.z, b.w);
      const double rad = hm_sqrt_fast(-2.0 * hm_log_unit(u1));
      hm_sincos2pi(u2, &sn[h], &cs[h]);
      z[h][0] = rad * cs[h]; z[h][1] = rad * sn[h];
      if constexpr (P >= 3) {
        // general p: Box-Muller pair k of object i comes from draw 1 + k (z_{2k}, z_{2k+1}); an odd p drops the last sine
        static_assert(P < 3 || ZD >= P, "z needs room for all p normals");
#pragma unroll
        for (int k = 1; 2 * k < P; ++k) {
          const U4 b2 = stream(seed, KIND_PLATE, (uint64_t)(i0 + h), t, 1u + (uint32_t)k);
          const double v1 = u01(b2.x, b2.y), v2 = u01(b2.z, b2.w);
          const double rad2 = hm_sqrt_fast(-2.0 * hm_log_unit(v1));
          double s2_, c2_;
          hm_sincos2pi(v2, &s2_, &c2_);
          z[h][2 * k] = rad2 * c2_;
          if (2 * k + 1 < P) z[h][2 * k + 1] = rad2 * s2_;
        }
      }
    }
  }
}
template <int P, int ZD, class KEY>
__device__ __forceinline__ void pair_draws(const KEY& seed, long long i0, uint32_t t, float (*z)[ZD], float* cs,
                                           float* sn, float* u) {
  static_assert(P <= 2, "fp32 state: p <= 2");
  if (P == 1) {
    const U4 r = stream(seed, KIND_PLATE, (uint64_t)i0 >> 1, t, 0u);
    const float u1 = u01f(r.x), u2 = u01f(r.y);
    u[0] = u01f(r.z); u[1] = u01f(r.w);
    const float rad = hm_sqrt_pos(-2.0f * logf(u1));
    float s_, c_;
    sincospif(2.0f * u2, &s_, &c_);
    z[0][0] = rad * c_; z[1][0] = rad * s_;
    z[0][1] = 0.0f; z[1][1] = 0.0f;
    cs[0] = cs[1] = 0.0f; sn[0] = sn[1] = 0.0f;
  } else {
#pragma unroll
    for (int h = 0; h < 2; ++h) {                  // per object: x -> u1, y -> u2, z -> accept uniform
      const U4 r = stream(seed, KIND_PLATE, (uint64_t)(i0 + h), t, 0u);
      const float u1 = u01f(r.x), u2 = u01f(r.y);
      u[h] = u01f(r.z);
      const float rad = hm_sqrt_pos(-2.0f * logf(u1));
      sincospif(2.0f * u2, &sn[h], &cs[h]);
      z[h][0] = rad * cs[h]; z[h][1] = rad * sn[h];
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// The sweep.  Fixed thread -> object map: at step k the thread with global index gid owns the VEC
// consecutive objects starting at VEC*(k*nthreads + gid): unit-stride 16-byte loads/stores per column.

// per-iteration constants of the sweep, in registers
template <class T> struct SweepCtx {
  uint32_t t;
  ThetaK kc, kp;
  KT<T> kT;
  T mcT[MC_N];
  T eta, astar;
  bool do_mom;
  double inv_k;
};
template <class T>
__device__ __forceinline__ SweepCtx<T> make_ctx(const Params& P, const Iter& it, const long long t_or_neg = -1) {
  SweepCtx<T> c;
  const long long t_it = t_or_neg >= 0 ? t_or_neg : it.t;       // (a kernel that starts before the tail has bumped it.t passes t)
  c.t = (uint32_t)t_it;
  c.kc = it.kc; c.kp = it.kp;
  c.kT = narrow<T>(c.kc);
#pragma unroll
  for (int j = 0; j < MC_N; ++j) c.mcT[j] = (T)P.mc[j];
  c.eta = (T)it.dr[slot3(t_it)].eta; c.astar = (T)P.astar_chi;
  c.do_mom = P.tail.keep_moments && t_it > P.tail.burn_in;
  c.inv_k = it.inv_k;
  return c;
}

// RAM steps 1-3 + population terms + moments for the VEC objects base .. base+VEC-1 held in x, l (updated in
// place; the caller stores them) and d.  acc = {S, Delta, n_accept, n_nonfinite} of this thread.
// The draws of ONE object (fp64, p >= 2), for the one-object-per-thread map of k_resident_gen: the accept uniform from its
// half of the pair's draw 0, its own normals from draws 1 + k -- the same words and values as pair_draws gives that object.
template <int P, int ZD, class KEY>
__device__ __forceinline__ void single_draws(const KEY& seed, long long i, uint32_t t, double* z, double* cs, double* sn, double* u) {
  static_assert(P >= 2 && ZD >= P, "single-object draws exist for p >= 2 (for p = 1 a pair shares one Box-Muller evaluation)");
  const U4 a = stream(seed, KIND_PLATE, (uint64_t)i >> 1, t, 0u);
  *u = (i & 1) ? u01(a.z, a.w) : u01(a.x, a.y);
  const U4 b = stream(seed, KIND_PLATE, (uint64_t)i, t, 1u);
  const double u1 = u01(b.x, b.y), u2 = u01(b.z, b.w);
  const double rad = hm_sqrt_fast(-2.0 * hm_log_unit(u1));
  hm_sincos2pi(u2, sn, cs);
  z[0] = rad * *cs; z[1] = rad * *sn;
#pragma unroll
  for (int k = 1; 2 * k < P; ++k) {
    const U4 b2 = stream(seed, KIND_PLATE, (uint64_t)i, t, 1u + (uint32_t)k);
    const double v1 = u01(b2.x, b2.y), v2 = u01(b2.z, b2.w);
    const double rad2 = hm_sqrt_fast(-2.0 * hm_log_unit(v1));
    double s2_, c2_;
    hm_sincos2pi(v2, &s2_, &c2_);
    z[2 * k] = rad2 * c2_;
    if (2 * k + 1 < P) z[2 * k + 1] = rad2 * s2_;
  }
}

// The plate draws of the VEC objects one thread owns at one step (theta- and chi-independent: a function of
// (seed, object, t) only, so they can be made ahead of the sweep -- k_persistent stages them in shared memory
// while the exchange and the theta step are in flight).
template <int MODEL, class T, int VEC_ = VecOf<T>::n> struct DrawSet {
  static constexpr int p = ModelDims<MODEL>::p, VEC = VEC_, ZD = p < 2 ? 2 : p;
  // values kept per object when staged: the p normals, the unit vector (p = 2 only) and the accept uniform
  static constexpr int NZ = p, NU = (p == 2 ? 2 : 0), NV = VEC * (NZ + NU + 1);
  T zz[VEC][ZD], csv[VEC], snv[VEC], uu[VEC];
  __device__ __forceinline__ void make(const Params& P, const long long base, const uint32_t t) {
    // KEY of the plate streams: the seed (fp64 kernels) or its ready-made round keys (fp32 kernels: philox.cuh; measured
    // -1.4 % on C4, while the fp64 kernels, bound by their fp64 chains, gain nothing or lose to the changed schedule)
    if constexpr (VEC == 1) {                 // one object per thread (k_resident_gen, small p >= 2 populations in fp64)
      single_draws<p, ZD>((uint64_t)P.tail.seed, P.obj_offset + base, t, zz[0], &csv[0], &snv[0], &uu[0]);
    } else {
#pragma unroll
      for (int v = 0; v < VEC; v += 2) {
        if constexpr (sizeof(T) == 4) pair_draws<p, ZD>(P.rk, P.obj_offset + base + v, t, &zz[v], &csv[v], &snv[v], &uu[v]);
        else pair_draws<p, ZD>((uint64_t)P.tail.seed, P.obj_offset + base + v, t, &zz[v], &csv[v], &snv[v], &uu[v]);
      }
    }
  }
  // staged layout: value q of thread-slot j at st[q * stride + j] (unit stride across a warp: conflict-free)
  __device__ __forceinline__ void put(T* st, const int stride) const {
    int q = 0;
#pragma unroll
    for (int v = 0; v < VEC; ++v) {
#pragma unroll
      for (int k = 0; k < NZ; ++k) st[(q++) * stride] = zz[v][k];
      if (NU) { st[(q++) * stride] = csv[v]; st[(q++) * stride] = snv[v]; }
      st[(q++) * stride] = uu[v];
    }
  }
  __device__ __forceinline__ void get(const T* st, const int stride) {
    int q = 0;
#pragma unroll
    for (int v = 0; v < VEC; ++v) {
#pragma unroll
      for (int k = 0; k < ZD; ++k) zz[v][k] = T(0);
#pragma unroll
      for (int k = 0; k < NZ; ++k) zz[v][k] = st[(q++) * stride];
      if (NU) { csv[v] = st[(q++) * stride]; snv[v] = st[(q++) * stride]; } else { csv[v] = T(0); snv[v] = T(0); }
      uu[v] = st[(q++) * stride];
    }
  }
};

// Running moments of object i's new chi (Welford; PAPER.md:337-341 reports posterior means and standard deviations of the
// member properties): mean += (x - mean)/k, M2 += (x - mean_old)(x - mean_new), with 1/k from the tail (Iter::inv_k).
template <int p, class T, int VEC>
__device__ __forceinline__ void moments_update(const Params& P, const SweepCtx<T>& c, const long long i, const T (*x)[VEC], const int v) {
#pragma unroll
  for (int j = 0; j < p; ++j) {
    const long long q = j * P.Npad + i;
    const double xv = (double)x[j][v];
    const double m0 = P.mom_mean[q];
    const double dl = xv - m0;
    const double m1 = m0 + dl * c.inv_k;
    P.mom_mean[q] = m1;
    P.mom_M2[q] += dl * (xv - m1);
  }
}
// Where the update sits.  Inside the per-object loop the compiler turns `if (do_mom)` into predication, so a run WITHOUT
// moments still issues the 14 instructions per object and component, predicated off: 9 % of the issue slots of the fp32
// kernel (ncu, C4), which is issue-bound -- there the update of all of a thread's objects sits behind ONE warp-uniform
// branch after the loop (C4 60.0 -> 57.2 us, same-box A/B).  The fp64 kernels are latency-bound, the slots are free, and
// the p = 2 kernel at its 128-register cap spills more with the late placement (C3 21.9 -> 22.25 us): they keep it inside.
template <class T> struct MomentsAfterLoop { static constexpr bool value = sizeof(T) == 4; };

// HOLD: the variant for frozen members.  An object whose mask byte is 0 takes no RAM step (chi, L and its
// update count stay bit for bit; its draws are made and discarded, the streams being counter-based) but still contributes
// a_i, b_i; with a per-object counter eta_n comes from the object's own update count n_i = count + 2.
// LateKp (k_persistent_dt): theta' and its constants are still being derived by the tail warps when the sweep of the next
// iteration starts; the population term at theta' reads them from shared memory, after a one-off wait per iteration.
struct LateKp {
  const ThetaK* kp;      // it.kp in shared memory
  int* wait;             // != 0: sync on BAR_THETAP (n threads) before the first use, then cleared
  int n;
};
template <int MODEL, class T, bool TAP, bool HOLD = false, bool LATE = false, int VEC_ = VecOf<T>::n, bool NO_MOM = false>
__device__ __forceinline__ void update_vec(const Params& P, const SweepCtx<T>& c, const long long base,
                                           T (*x)[VEC_], T (*l)[VEC_], const T (*d)[VEC_], double* sum,
                                           const DrawSet<MODEL, T, VEC_>* staged = nullptr, const LateKp* late = nullptr) {
  constexpr int p = ModelDims<MODEL>::p, ntri = p * (p + 1) / 2, ncols = ModelDims<MODEL>::ncols;
  constexpr int VEC = VEC_;
  DrawSet<MODEL, T, VEC_> ds_;
  if (!staged) ds_.make(P, base, c.t);
  const DrawSet<MODEL, T, VEC_>& ds = staged ? *staged : ds_;
  const T (*zz)[DrawSet<MODEL, T, VEC_>::ZD] = ds.zz;
  const T* csv = ds.csv; const T* snv = ds.snv; const T* uu = ds.uu;
#pragma unroll
  for (int v = 0; v < VEC; ++v) {
    const long long i = base + v;
    const bool live = i < P.N;
    bool upd = true;
    T eta_v = c.eta;
    if constexpr (HOLD) {
      if (live && P.mask) upd = P.mask[i] != 0;
      if (live && upd && P.cnt) {
        const unsigned n_i = P.cnt[i];
        P.cnt[i] = n_i + 1u;
        // the common case (updated in every iteration so far) reuses the iteration's eta; same function, same argument
        if (c.eta != T(0) && n_i + 1u != c.t) eta_v = (T)pow((double)n_i + 2.0, -P.tail.eta_exp);
      }
    }
    T xi[p], di[ncols];
    const T cs = csv[v], sn = snv[v], u = uu[v];
    const T* z = zz[v];
#pragma unroll
    for (int j = 0; j < p; ++j) xi[j] = x[j][v];
#pragma unroll
    for (int q = 0; q < ncols; ++q) di[q] = d[q][v];
    // step 1: chi' = chi + L z
    T yi[p];
#pragma unroll
    for (int r = 0; r < p; ++r) {
      T a_ = xi[r];
#pragma unroll
      for (int k = 0; k <= r; ++k) a_ += l[r * (r + 1) / 2 + k][v] * z[k];
      yi[r] = a_;
    }
    // step 2: alpha = min{1, pi(chi')/pi(chi)}
    using PL = Plate<MODEL, T>;
    const typename PL::Pt qc = PL::point(xi), qp = PL::point(yi);
    const T pc = PL::target(qc, di, c.kT, c.mcT), pp = PL::target(qp, di, c.kT, c.mcT);
    const T diff = pp - pc;
    const bool bad = diff != diff;
    const T la = bad ? T(-INFINITY) : (diff < T(0) ? diff : T(0));
    const T alpha = hm_exp_nonpos(la);
    const bool acc = HOLD ? (upd && u < alpha) : (u < alpha);
    const typename PL::Pt qn = acc ? qp : qc;
#pragma unroll
    for (int j = 0; j < p; ++j) x[j][v] = acc ? yi[j] : xi[j];
    // step 3: L <- L chol(I + c uu^T), u = z/|z| = (cs, sn)
    const T cc = eta_v * (alpha - c.astar);
    T ln[ntri];
    if constexpr (p == 1) {
      ln[0] = l[0][v] * hm_sqrt_pos(T(1) + cc);
    } else if constexpr (p >= 3) {
      // general p, the rank-one update in closed form (theta_step.cuh::ram_coeffs): with u = z/|z| and
      // s_j = 1 + c sum_{k<j} u_k^2:  K = chol(I + c u u^T) has K_jj = sqrt(s_{j+1}/s_j), K_ij = c u_i u_j/sqrt(s_j s_{j+1}),
      // and (L K)_ij = L_ij K_jj + (c u_j/sqrt(s_j s_{j+1})) sum_{k=j+1..i} L_ik u_k -- the unique left factor of Eq. 2.6
      T n2 = T(0);
#pragma unroll
      for (int j = 0; j < p; ++j) n2 += z[j] * z[j];
      const T rn = hm_rsqrt(n2);
      T uh[p], sj[p + 1];
      T run = T(0);
      sj[0] = T(1);
#pragma unroll
      for (int j = 0; j < p; ++j) { uh[j] = z[j] * rn; run += uh[j] * uh[j]; sj[j + 1] = T(1) + cc * run; }
#pragma unroll
      for (int j = 0; j < p; ++j) {
        const T rr = hm_rsqrt(sj[j] * sj[j + 1]);
        const T Kd = sj[j + 1] * rr, g = cc * uh[j] * rr;
#pragma unroll
        for (int i = j; i < p; ++i) {
          T W = T(0);
#pragma unroll
          for (int k = j + 1; k <= i; ++k) W += l[i * (i + 1) / 2 + k][v] * uh[k];
          ln[i * (i + 1) / 2 + j] = l[i * (i + 1) / 2 + j][v] * Kd + g * W;
        }
      }
    } else {
      const T s1 = T(1) + cc * cs * cs;
      T k00, ik00;
      hm_sqrt_both(s1, &k00, &ik00);                       // sqrt(s1), 1/sqrt(s1): no division in the update
      const T k10 = cc * cs * sn * ik00;
      const T k11 = hm_sqrt_pos(T(1) + cc) * ik00;
      ln[0] = l[0][v] * k00;
      ln[1] = l[1][v] * k00 + l[2][v] * k10;
      ln[2] = l[2][v] * k11;
    }
    // population terms at the new chi, fp64
    if constexpr (LATE) {
      if (*late->wait) { bar_sync(BAR_THETAP, late->n); *late->wait = 0; }
    }
    const double a = PL::pop(qn, di, c.kc, P.mc), b = PL::pop(qn, di, LATE ? *late->kp : c.kp, P.mc);
    if (live) {
      if constexpr (HOLD) {
#pragma unroll
        for (int k = 0; k < ntri; ++k) ln[k] = upd ? ln[k] : l[k][v];
      }
#pragma unroll
      for (int k = 0; k < ntri; ++k) l[k][v] = ln[k];
      sum[0] += a; sum[1] += b - a;
      sum[2] += acc ? 1.0 : 0.0; sum[3] += (bad && upd) ? 1.0 : 0.0;
      if constexpr (!MomentsAfterLoop<T>::value && !NO_MOM) {
        if (c.do_mom) moments_update<p, T, VEC>(P, c, i, x, v);
      }
      if (TAP) {
        const DevTaps& tp = P.taps;
#pragma unroll
        for (int j = 0; j < p; ++j) if (tp.chi_prop) tp.chi_prop[j * P.N + i] = (double)(upd ? yi[j] : xi[j]);
        if (tp.pi_cur) tp.pi_cur[i] = (double)pc + tp.shift_c;
        if (tp.pi_prop) tp.pi_prop[i] = (double)(upd ? pp : pc) + tp.shift_c;
        if (tp.alpha) tp.alpha[i] = upd ? (double)alpha : 0.0;
        if (tp.u) tp.u[i] = upd ? (double)u : 1.0;
        if (tp.accepted) tp.accepted[i] = acc ? 1 : 0;
#pragma unroll
        for (int k = 0; k < ntri; ++k) if (tp.L_new) tp.L_new[k * P.N + i] = (double)ln[k];
        if (tp.a) tp.a[i] = a + tp.shift_c;
        if (tp.b) tp.b[i] = b + tp.shift_p;
      }
    } else {
#pragma unroll
      for (int j = 0; j < p; ++j) x[j][v] = xi[j];
    }
  }
  if constexpr (MomentsAfterLoop<T>::value && !NO_MOM) {
    if (c.do_mom) {
#pragma unroll
      for (int v = 0; v < VEC; ++v)
        if (base + v < P.N) moments_update<p, T, VEC>(P, c, base + v, x, v);
    }
  }
}

// selection-integral slice (M1): term k belongs to block k % gridDim.x, thread k / gridDim.x
template <int MODEL>
__device__ __forceinline__ double selection_slice(const Params& P, const ThetaK& kp, const int sweep_threads) {
  double tq = 0.0;
  if (has_selection(MODEL) && !P.tail.freeze_theta) {
    for (int k = (int)blockIdx.x + (int)gridDim.x * (int)threadIdx.x; k < NQUAD; k += (int)gridDim.x * sweep_threads)
      tq += selection_term<MODEL>(kp, P.qW[k], P.qx[k], P.qex[k]);
  }
  return tq;
}

// one step of the sweep: load the thread's VEC objects, update, store
template <int MODEL, class T, bool TAP, bool HOLD = false, bool LATE = false, bool NO_MOM = false>
__device__ __forceinline__ void sweep_step(const Params& P, const SweepCtx<T>& c, const long long base, double* acc,
                                           const DrawSet<MODEL, T>* staged, const LateKp* late = nullptr) {
  constexpr int p = ModelDims<MODEL>::p, ntri = p * (p + 1) / 2, ncols = ModelDims<MODEL>::ncols;
  constexpr int VEC = VecOf<T>::n;
  const long long Npad = P.Npad;
  T* const chi = static_cast<T*>(P.chi);
  T* const Lm = static_cast<T*>(P.L);
  const T* const dat = static_cast<const T*>(P.data);
  T x[p][VEC], l[ntri][VEC], d[ncols][VEC];
#pragma unroll
  for (int j = 0; j < p; ++j) ld_vec<T>(chi + j * Npad + base, x[j], false);
#pragma unroll
  for (int k = 0; k < ntri; ++k) ld_vec<T>(Lm + k * Npad + base, l[k], false);
#pragma unroll
  for (int cc = 0; cc < ncols; ++cc) ld_vec<T>(dat + cc * Npad + base, d[cc], true);
  update_vec<MODEL, T, TAP, HOLD, LATE, VecOf<T>::n, NO_MOM>(P, c, base, x, l, d, acc, staged, late);
#pragma unroll
  for (int j = 0; j < p; ++j) st_vec(chi + j * Npad + base, x[j]);
#pragma unroll
  for (int k = 0; k < ntri; ++k) st_vec(Lm + k * Npad + base, l[k]);
}

// L2 prefetch of the columns of the step that starts at object `base` (no registers held, unlike a load issued early)
#ifndef HM_PREFETCH
#define HM_PREFETCH 1
#endif
template <int MODEL, class T>
__device__ __forceinline__ void prefetch_step(const Params& P, const long long base) {
#if HM_PREFETCH
  constexpr int p = ModelDims<MODEL>::p, ntri = p * (p + 1) / 2, ncols = ModelDims<MODEL>::ncols;
  const long long Npad = P.Npad;
  const T* const chi = static_cast<const T*>(P.chi);
  const T* const Lm = static_cast<const T*>(P.L);
  const T* const dat = static_cast<const T*>(P.data);
#pragma unroll
  for (int j = 0; j < p; ++j) asm volatile("prefetch.global.L2 [%0];" ::"l"(chi + j * Npad + base));
#pragma unroll
  for (int k = 0; k < ntri; ++k) asm volatile("prefetch.global.L2 [%0];" ::"l"(Lm + k * Npad + base));
#pragma unroll
  for (int cc = 0; cc < ncols; ++cc) asm volatile("prefetch.global.L2 [%0];" ::"l"(dat + cc * Npad + base));
#endif
}

// part[NPART] receives this thread's partial sums in ascending object order.  stage / n_stage: the plate draws of
// the thread's first n_stage steps, made ahead by stage_draws (k_persistent); the same values bit for bit.
template <int MODEL, class T, bool TAP, bool AHEAD = false, bool HOLD = false>
__device__ __forceinline__ void sweep(const Params& P, const Iter& it, double* part, const T* stage = nullptr,
                                      const int n_stage = 0, const bool prefetch = false) {
  constexpr int VEC = VecOf<T>::n;
  const long long N = P.N;
  const long long nthreads = (long long)gridDim.x * blockDim.x;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const SweepCtx<T> c = make_ctx<T>(P, it);
  double acc[4] = {0.0, 0.0, 0.0, 0.0};
  long long base = (long long)VEC * gid;
  const long long stride = (long long)VEC * nthreads;
  if constexpr (AHEAD) {
    // while a step is computed the next one is on its way from HBM to L2 (after the last step: the first step of
    // the next iteration, which then arrives during the exchange and the theta step)
    const int B = (int)blockDim.x;
    for (int s = 0; s < n_stage && base < N; ++s, base += stride) {
      if (prefetch) prefetch_step<MODEL, T>(P, base + stride < N ? base + stride : (long long)VEC * gid);
      DrawSet<MODEL, T> ds;
      ds.get(stage + (size_t)s * DrawSet<MODEL, T>::NV * B + threadIdx.x, B);
      sweep_step<MODEL, T, TAP>(P, c, base, acc, &ds);
    }
    for (; base < N; base += stride) {
      if (prefetch) prefetch_step<MODEL, T>(P, base + stride < N ? base + stride : (long long)VEC * gid);
      sweep_step<MODEL, T, TAP>(P, c, base, acc, nullptr);
    }
  } else {
    for (; base < N; base += stride) sweep_step<MODEL, T, TAP, HOLD>(P, c, base, acc, nullptr);
  }
  part[0] = acc[0]; part[1] = acc[1]; part[2] = selection_slice<MODEL>(P, c.kp, (int)blockDim.x); part[3] = acc[2]; part[4] = acc[3];
}

// Stage the plate draws of iteration t for the first n_stage steps of every thread of this block.  Called by the
// `nworkers` threads with worker index w = 0 .. nworkers-1 (the warps that do not run the theta tail).
template <int MODEL, class T>
__device__ __forceinline__ void stage_draws(const Params& P, const uint32_t t, T* stage, const int n_stage, const int w,
                                            const int nworkers) {
  constexpr int VEC = VecOf<T>::n;
  const int B = (int)blockDim.x;
  const long long nthreads = (long long)gridDim.x * B;
  for (int idx = w; idx < n_stage * B; idx += nworkers) {
    const int s = idx / B, j = idx - s * B;
    const long long base = (long long)VEC * ((long long)s * nthreads + (long long)blockIdx.x * B + j);
    if (base < P.N) {
      DrawSet<MODEL, T> ds;
      ds.make(P, base, t);
      ds.put(stage + (size_t)s * DrawSet<MODEL, T>::NV * B + j, B);
    }
  }
}

// Deterministic block reduction of NQ quantities: shuffle tree inside each warp, then warp 0 over the per-warp
// results.  Returns the block totals in v[] of thread 0.  red: shared [32][NPART].
template <int NQ>
__device__ __forceinline__ void block_reduce(double* v, double (*red)[NPART]) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) v[q] += __shfl_down_sync(0xffffffffu, v[q], o);
  }
  if (lane == 0) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) red[wid][q] = v[q];
  }
  __syncthreads();
  if (wid == 0) {
    double w[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) w[q] = lane < nw ? red[lane][q] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
      for (int q = 0; q < NQ; ++q) w[q] += __shfl_down_sync(0xffffffffu, w[q], o);
    }
#pragma unroll
    for (int q = 0; q < NQ; ++q) v[q] = w[q];
  }
}

// Same tree, but EVERY warp redoes the second stage, so every thread of the block ends up with the totals
// (no broadcast barrier before the mailbox push).
template <int NQ>
__device__ __forceinline__ void block_reduce_all(double* v, double (*red)[NPART]) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) v[q] += __shfl_down_sync(0xffffffffu, v[q], o);
  }
  if (lane == 0) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) red[wid][q] = v[q];
  }
  __syncthreads();
#pragma unroll
  for (int q = 0; q < NQ; ++q) v[q] = lane < nw ? red[lane][q] : 0.0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) v[q] += __shfl_down_sync(0xffffffffu, v[q], o);
  }
#pragma unroll
  for (int q = 0; q < NQ; ++q) v[q] = __shfl_sync(0xffffffffu, v[q], 0);
}

// Fixed-order sum over blocks by warp 0: lane l adds blocks l, l+32, ... in order, then a shuffle tree; the
// result is broadcast to every lane.  Both slot formats below use exactly this order, so the persistent
// kernel and the k_sweep + k_tail pair produce the same bits.
template <int NQ>
__device__ __forceinline__ void lanes_to_total(double* v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) v[q] += __shfl_down_sync(0xffffffffu, v[q], o);
  }
#pragma unroll
  for (int q = 0; q < NQ; ++q) v[q] = __shfl_sync(0xffffffffu, v[q], 0);
}

// plain slots [nblocks][NPART] written by k_sweep (a kernel boundary orders them)
__device__ __forceinline__ void slots_reduce(const double* slots, int nblocks, double* tot) {
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int q = 0; q < NPART; ++q) tot[q] = 0.0;
  for (int g = lane; g < nblocks; g += 32) {
#pragma unroll
    for (int q = 0; q < NPART; ++q) tot[q] += __ldcg(slots + (size_t)g * NPART + q);
  }
  lanes_to_total<NPART>(tot);
}

// Per-iteration exchange of the persistent kernel: the grid-wide reduction AND the barrier in one round trip.
// Every block has a private mailbox with one slot per block; a block PUSHES its two partials (Delta, Tq) into
// its slot of every mailbox (thread r writes to reader r: one 16-byte store per thread and value), and warp 0
// of a block polls only its own mailbox.  No line is ever polled by more than one SM, so nothing queues at L2
// (an all-read-all layout measured 4 us from last publish to visibility; profiles/r01b).  A slot holds, per
// value, two 8-byte words {epoch << 32 | 32 data bits}: an 8-byte store is single-copy atomic, so a reader that
// sees the right epoch in a word has that word's data -- no fence, no arrival counter, no second read.  Mailboxes
// alternate by iteration parity: a block can be at most one iteration ahead of the slowest reader (it needs
// everybody's slot of iteration k to get past k).  Epochs increase over the sampler's lifetime.
//   mbox layout: [parity][reader][value 0..MBOX_NV-1][writer][2 words]; a kernel uses the first NV values
constexpr int MBOX_NV = 3;
__device__ __forceinline__ size_t mbox_parity_words(int G) { return (size_t)2 * MBOX_NV * G * G; }
__device__ __forceinline__ size_t mbox_reader_words(int G) { return (size_t)2 * MBOX_NV * G; }
template <int NV>
__device__ __forceinline__ void mbox_push(unsigned long long* mbox_parity, int G, int writer, unsigned epoch, const double* val,
                                          int first, int stride) {
  const unsigned long long e = (unsigned long long)epoch << 32;
  unsigned long long w0[NV], w1[NV];
#pragma unroll
  for (int q = 0; q < NV; ++q) {
    const unsigned long long u = (unsigned long long)__double_as_longlong(val[q]);
    w0[q] = e | (u & 0xffffffffull); w1[q] = e | (u >> 32);
  }
  for (int r = first; r < G; r += stride) {
    unsigned long long* box = mbox_parity + (size_t)r * mbox_reader_words(G);
#pragma unroll
    for (int q = 0; q < NV; ++q)
      asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(box + 2 * q * G + 2 * writer), "l"(w0[q]), "l"(w1[q]) : "memory");
  }
}
// Collect (warp 0): lane l owns writers l, l+32, ...; up to LL_BATCH of them are polled TOGETHER (independent
// loads in flight: one L2 round trip once everything has arrived), then added in ascending order.
constexpr int LL_BATCH = 5;   // ceil(148 / 32): the whole one-block-per-SM grid in one batch
template <int NV>
__device__ __forceinline__ void mbox_collect(const unsigned long long* box, int G, unsigned epoch, double* tot) {
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int q = 0; q < NV; ++q) tot[q] = 0.0;
  for (int g0 = lane; g0 < G; g0 += 32 * LL_BATCH) {
    unsigned long long w[LL_BATCH][2 * NV];
    bool ok;
    do {
      ok = true;
#pragma unroll
      for (int j = 0; j < LL_BATCH; ++j) {
        const int g = g0 + 32 * j;
        if (g < G) {
#pragma unroll
          for (int q = 0; q < NV; ++q)
            asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(w[j][2 * q]), "=l"(w[j][2 * q + 1]) : "l"(box + 2 * q * G + 2 * g) : "memory");
        }
      }
#pragma unroll
      for (int j = 0; j < LL_BATCH; ++j) {
        if (g0 + 32 * j < G) {
#pragma unroll
          for (int q = 0; q < 2 * NV; ++q) ok = ok && (unsigned)(w[j][q] >> 32) == epoch;
        }
      }
    } while (!ok);
#pragma unroll
    for (int j = 0; j < LL_BATCH; ++j) {
      if (g0 + 32 * j < G) {
#pragma unroll
        for (int q = 0; q < NV; ++q)
          tot[q] += __longlong_as_double((long long)((w[j][2 * q] & 0xffffffffull) | (w[j][2 * q + 1] << 32)));
      }
    }
  }
  lanes_to_total<NV>(tot);
}

__device__ __forceinline__ void copy_iter(Iter* dst, const Iter* src) {
  const int n = (int)(sizeof(Iter) / sizeof(double));
  const double* s = reinterpret_cast<const double*>(src);
  double* d = reinterpret_cast<double*>(dst);
  for (int k = threadIdx.x; k < n; k += blockDim.x) d[k] = s[k];
}
static_assert(sizeof(Iter) % sizeof(double) == 0, "Iter is copied as doubles");

// ---------------------------------------------------------------------------------------------------
// THETA_DEVICE_TAIL: the whole Gibbs loop in one cooperative launch (co-residency of all blocks is what the
// flag exchange needs).  Per iteration: sweep -> block partials -> flagged slot -> warp 0 of EVERY block collects
// all slots in the same fixed order -> block-parallel theta tail (identical in every block) -> next sweep.
// One grid-wide round trip per iteration.  Accept / non-finite counters stay in registers until the launch ends.
// AHEAD: the variant that works ahead of the exchange -- plate draws of the next iteration staged in shared memory by
// the warps that do not run the theta tail, next step's columns prefetched into L2.  The plain variant
// is kept for the populations that gain nothing from either (p = 2 out of L2: C3).  Same chain bit for bit.
enum : int { PK_PLAIN = 0, PK_AHEAD = 1, PK_HOLD = 2 };   // PK_HOLD: the plain kernel with the frozen-member hooks of update_vec
template <int MODEL, class T, int BLOCK, int VARIANT>
__global__ void __launch_bounds__(BLOCK, 1) k_persistent(const Params P, const long long n_iter, const unsigned epoch0,
                                                         const int n_stage, const int prefetch) {
  constexpr bool AHEAD = VARIANT == PK_AHEAD, HOLD = VARIANT == PK_HOLD;
  __shared__ Iter it;
  __shared__ double red[32][NPART];
  extern __shared__ __align__(16) unsigned char stage_raw[];   // n_stage x DrawSet::NV x BLOCK values of T
  T* const stage = reinterpret_cast<T*>(stage_raw);
  constexpr int TAILT = 128;                                   // the four warps of the theta tail
  copy_iter(&it, P.iter);
  __syncthreads();
  // draws of the launch's first iteration: every thread stages (nothing to overlap with yet)
  if (AHEAD) {
    stage_draws<MODEL, T>(P, (uint32_t)it.t, stage, n_stage, (int)threadIdx.x, BLOCK);
    __syncthreads();
  }
  const int G = (int)gridDim.x;
  double cnt[2] = {0.0, 0.0};
  for (long long k = 0; k < n_iter; ++k) {
    double part[NPART];
    const uint32_t t_next = (uint32_t)it.t + 1u;
    sweep<MODEL, T, false, AHEAD, HOLD>(P, it, part, stage, n_stage, prefetch != 0);
    cnt[0] += part[3]; cnt[1] += part[4];
    double dq[2] = {part[1], part[2]};
    block_reduce_all<2>(dq, red);
    constexpr int NVX = has_selection(MODEL) ? 2 : 1;   // only M1 / M4 have a selection-integral slice to exchange
    unsigned long long* mb = P.mbox + (size_t)(k & 1) * mbox_parity_words(G);
    const unsigned epoch = epoch0 + (unsigned)k;
    mbox_push<NVX>(mb, G, (int)blockIdx.x, epoch, dq, (int)threadIdx.x, (int)blockDim.x);
    // warps 0-3: collect + theta tail (the serial chain); the other warps meanwhile make the plate draws of the
    // first n_stage steps of iteration t + 1, which depend on nothing but (seed, object, t + 1)
    if (threadIdx.x < TAILT) {
      double tot[NPART] = {0.0, 0.0, 0.0, 0.0, 0.0};
      if (threadIdx.x < 32) {
        double t2[2] = {0.0, 0.0};
        mbox_collect<NVX>(mb + (size_t)blockIdx.x * mbox_reader_words(G), G, epoch, t2);
        tot[1] = t2[0]; tot[2] = t2[1];
      }
      tail_block<MODEL>(it, P.tail, tot, blockIdx.x == 0 ? P.trace : nullptr, (int)(threadIdx.x >> 5), SyncNamed<1, TAILT>());
    } else if (AHEAD && k + 1 < n_iter) {
      stage_draws<MODEL, T>(P, t_next, stage, n_stage, (int)threadIdx.x - TAILT, BLOCK - TAILT);
    }
    __syncthreads();                    // the plain variant's other warps wait here: only warps 0-3 run the tail
  }
  block_reduce<2>(cnt, red);
  if (threadIdx.x == 0) {
    P.blk_cnt[2 * blockIdx.x] += (unsigned long long)cnt[0];
    P.blk_cnt[2 * blockIdx.x + 1] += (unsigned long long)cnt[1];
  }
  if (blockIdx.x == 0) copy_iter(P.iter, &it);
}

// The streaming kernel with DEDICATED tail warps: SWEEP sweep threads + 4 tail warps per block.
// The sweep warps hand their partials over and wait only for the DECISION of the theta step (theta_{t+1} and its constants);
// the rest of the tail -- RAM update of L_theta, theta', its constants, prior, W: ~4,000 cycles -- runs on the tail warps
// while the sweep warps already load, draw, propose and decide the first objects of iteration t + 1; the population term at
// theta' waits once per iteration for the tail to finish (LateKp).  Worth it where fewer sweep warps with more registers are
// as fast as 16 (p = 2 in fp64: the sweep is latency-bound); same per-object arithmetic, its own (fixed) summation order.
// NO_MOM: the instantiation for handles that keep no running moments (cfg.keep_chi_moments = 0).  As a run-time flag the
// Welford update stays in the code, predicated off, and holds address registers in a kernel that sits at its register cap.
constexpr int DT_TAIL = 128;
template <int MODEL, class T, int SWEEP, bool NO_MOM = false>
__global__ void __launch_bounds__(SWEEP + DT_TAIL, 1) k_persistent_dt(const Params P, const long long n_iter, const unsigned epoch0,
                                                                      const int n_stage, const int prefetch) {
  constexpr int VEC = VecOf<T>::n, THREADS = SWEEP + DT_TAIL, SW = SWEEP / 32, NV = DrawSet<MODEL, T>::NV;
  // a sweep thread makes the plate draws of its OWN first n_stage steps of iteration t + 1 while it waits for the decision of
  // iteration t (they depend on (seed, object, t + 1) only) and parks them in shared memory: [step][value][thread]
  extern __shared__ __align__(16) unsigned char stage_raw[];
  T* const stage = reinterpret_cast<T*>(stage_raw) + threadIdx.x;
  __shared__ Iter it;
  __shared__ double red[2][SW];
  __shared__ unsigned long long cnt_sm[2];
  const int tid = (int)threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int G = (int)gridDim.x;
  copy_iter(&it, P.iter);
  if (tid < 2) cnt_sm[tid] = 0ull;
  __syncthreads();
  const long long t0 = it.t;
  if (tid < SWEEP) {
    const long long N = P.N;
    const long long stride = (long long)VEC * G * SWEEP;
    const long long first = (long long)VEC * ((long long)blockIdx.x * SWEEP + tid);
    double nacc = 0.0, nnan = 0.0;
    auto stage_own = [&](const uint32_t t) {
      long long base = first;
      for (int s = 0; s < n_stage && base < N; ++s, base += stride) {
        DrawSet<MODEL, T> ds;
        ds.make(P, base, t);
        ds.put(stage + (size_t)s * NV * SWEEP, SWEEP);
      }
    };
    stage_own((uint32_t)t0);
    for (long long k = 0; k < n_iter; ++k) {
      if (k > 0) bar_sync(BAR_THETA, THREADS);               // the decision of iteration t - 1 is taken: kc, eta, moment count
      const SweepCtx<T> c = make_ctx<T>(P, it, t0 + k);      // (its kp is not used: LateKp)
      int wait = k > 0 ? 1 : 0;
      // the late wait inside update_vec is a block barrier and needs the warp converged there: a warp whose lanes do not ALL
      // own a first-step object (the ragged end of a small population) waits up front instead -- warp-uniform either way
      if (wait && !__all_sync(0xffffffffu, first < N)) { bar_sync(BAR_THETAP, THREADS); wait = 0; }
      const LateKp late{&it.kp, &wait, THREADS};
      double acc[4] = {0.0, 0.0, 0.0, 0.0};
      long long base = first;
      for (int s = 0; s < n_stage && base < N; ++s, base += stride) {
        if (prefetch) prefetch_step<MODEL, T>(P, base + stride < N ? base + stride : first);
        DrawSet<MODEL, T> ds;
        ds.get(stage + (size_t)s * NV * SWEEP, SWEEP);
        sweep_step<MODEL, T, false, false, true, NO_MOM>(P, c, base, acc, &ds, &late);
      }
      for (; base < N; base += stride) {
        if (prefetch) prefetch_step<MODEL, T>(P, base + stride < N ? base + stride : first);
        sweep_step<MODEL, T, false, false, true, NO_MOM>(P, c, base, acc, nullptr, &late);
      }
      if (wait) bar_sync(BAR_THETAP, THREADS);               // (not reached with wait set: kept as a guard)
      nacc += acc[2]; nnan += acc[3];
      double v = acc[1];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
      if (lane == 0) red[k & 1][warp] = v;
      // (no fence needed: when the barrier completes, bar.arrive has ordered this thread's prior shared-memory writes for its participants)
      bar_arrive(BAR_PARTIALS, THREADS);
      if (k + 1 < n_iter) stage_own((uint32_t)(t0 + k + 1));
    }
    bar_sync(BAR_THETA, THREADS);
    bar_sync(BAR_THETAP, THREADS);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      nacc += __shfl_down_sync(0xffffffffu, nacc, o);
      nnan += __shfl_down_sync(0xffffffffu, nnan, o);
    }
    if (lane == 0) {
      atomicAdd(&cnt_sm[0], (unsigned long long)nacc);
      atomicAdd(&cnt_sm[1], (unsigned long long)nnan);
    }
  } else {
    const int tw = warp - SW, ttid = tid - SWEEP;
    for (long long k = 0; k < n_iter; ++k) {
      bar_sync(BAR_PARTIALS, THREADS);
      double dq[1];
      dq[0] = lane < SW ? red[k & 1][lane] : 0.0;
      lanes_to_total<1>(dq);
      unsigned long long* mb = P.mbox + (size_t)(k & 1) * mbox_parity_words(G);
      const unsigned epoch = epoch0 + (unsigned)k;
      mbox_push<1>(mb, G, (int)blockIdx.x, epoch, dq, ttid, DT_TAIL);
      double tot[NPART] = {0.0, 0.0, 0.0, 0.0, 0.0};
      if (tw == 0) {
        double t1[1];
        mbox_collect<1>(mb + (size_t)blockIdx.x * mbox_reader_words(G), G, epoch, t1);
        tot[1] = t1[0];
      }
      tail_block<MODEL>(it, P.tail, tot, blockIdx.x == 0 ? P.trace : nullptr, tw, SyncNamed<BAR_TAIL, DT_TAIL>(),
                        ArriveNamed<BAR_THETA, THREADS>());
      // (no fence needed: when the barrier completes, bar.arrive has ordered this thread's prior shared-memory writes for its participants)
      bar_arrive(BAR_THETAP, THREADS);
    }
  }
  __syncthreads();
  if (tid == 0) {
    P.blk_cnt[2 * blockIdx.x] += cnt_sm[0];
    P.blk_cnt[2 * blockIdx.x + 1] += cnt_sm[1];
  }
  if (blockIdx.x == 0) copy_iter(P.iter, &it);
}

// One sweep as its own launch (THETA_GRAPH, THETA_HOST, debug_step).  Same grid, same maps, same order.
template <int MODEL, class T, int BLOCK, bool TAP, bool HOLD = false>
__global__ void __launch_bounds__(BLOCK, 1) k_sweep(const Params P) {
  __shared__ Iter it;
  __shared__ double red[32][NPART];
  copy_iter(&it, P.iter);
  __syncthreads();
  double part[NPART];
  sweep<MODEL, T, TAP, false, HOLD>(P, it, part);
  block_reduce<NPART>(part, red);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < NPART; ++q) P.slots[(size_t)blockIdx.x * NPART + q] = part[q];
  }
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
    if (has_selection(MODEL)) {
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
  if (P.cnt) P.cnt[i] = 0u;
}

}  // namespace hm
