// resident_gen.cuh -- the on-chip persistent Gibbs kernel for every (model, precision) the tuned p = 1 fp64 kernel of
// resident.cuh does not cover: p >= 2 in fp64 (M2, the normal-normal family p = 3 .. 6) and the fp32-state models.
// DESIGN.md section 8.5.
//
// Same idea as k_resident: a population that fits in shared memory stays there for the whole launch (chi, L, data columns:
// HBM / L2 are touched at launch start and end only), the theta-independent plate draws of iteration t + 1 are made while
// the exchange and the theta step of iteration t are in flight, and 4 dedicated warps run the exchange and the theta tail.
// The per-object arithmetic is update_vec itself (kernels.cuh), fed from shared memory and from draws staged there (it starts at
// the theta DECISION and reads theta' late, like k_persistent_dt), so the
// chain is the streaming kernels' to the last bit of every object; only the order in which block partials are added differs
// (fixed, so still deterministic).  The running chi moments stay in global memory (they are touched once per iteration).
#pragma once
#include "resident.cuh"

namespace hm {

// shared-memory values of T per object: the state and data columns plus the staged draws of one iteration
template <int MODEL, class T, int VEC_ = VecOf<T>::n> struct ResGenValues {
  static constexpr int p = ModelDims<MODEL>::p, ntri = p * (p + 1) / 2, ncols = ModelDims<MODEL>::ncols;
  static constexpr int VEC = VEC_, NV = DrawSet<MODEL, T, VEC_>::NV;
  static constexpr int n_state = p + ntri + ncols;
  static constexpr int n_values = n_state + NV / VEC;
};

// one group of VEC adjacent objects of a column: a 16-byte access for the full vector, a scalar one for VEC = 1
template <class T, int VEC>
__device__ __forceinline__ void rg_load(const T* q, T* out, bool ro) {
  if constexpr (VEC == VecOf<T>::n) ld_vec<T>(q, out, ro);
  else { static_assert(VEC == 1, "VEC is 1 or a full 16-byte vector"); out[0] = ro ? __ldg(q) : *q; }
}
template <class T, int VEC>
__device__ __forceinline__ void rg_store(T* q, const T* v) {
  if constexpr (VEC == VecOf<T>::n) st_vec(q, v);
  else *q = v[0];
}

// VEC_: objects per thread group.  The full 16-byte vector by default; 1 for populations of at most one object per sweep
// thread (N <= blocks x 256: C6), where an object PAIR per thread would leave half the sweep warps idle and every busy
// thread with twice the serial work (C6: update ~6,000 + draws ~3,600 cycles per iteration on 4 of 8 warps).
template <int MODEL, class T, int VEC_ = VecOf<T>::n>
__global__ void __launch_bounds__(RG_THREADS, 1) k_resident_gen(const Params P, const long long n_iter, const unsigned epoch0,
                                                                const int R, const int OB) {
  using V = ResGenValues<MODEL, T, VEC_>;
  using DS = DrawSet<MODEL, T, VEC_>;
  constexpr int p = V::p, ntri = V::ntri, ncols = V::ncols, VEC = V::VEC, NV = V::NV;
  extern __shared__ __align__(16) unsigned char sm_raw[];
  T* const sm = reinterpret_cast<T*>(sm_raw);
  __shared__ Iter it;
  __shared__ double red[2][RG_SW];
  __shared__ unsigned long long cnt_sm[2];
  const int tid = (int)threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const bool is_tail = warp >= RG_SW;
  const int G = (int)gridDim.x;
  const long long N = P.N, Npad = P.Npad;
  // A block owns the OB (a multiple of VEC) contiguous objects [blockIdx.x * OB, (blockIdx.x + 1) * OB); a sweep thread owns
  // groups of VEC adjacent objects: group g of thread tid starts at obj0 + g * VEC * RG_S.  R = VEC * (groups per thread).
  const long long obj0 = (long long)blockIdx.x * OB + (long long)VEC * tid;
  const long long obj_end = (long long)(blockIdx.x + 1) * OB < N ? (long long)(blockIdx.x + 1) * OB : N;
  const int ngroups = R / VEC;
  // state region [value][slot][thread], draw region [group][draw value][thread]: unit stride across a warp, conflict-free
  T* const st_my = sm + tid;
  T* const dr_my = sm + (size_t)V::n_state * R * RG_S + tid;
#define HM_GAT(v, s) st_my[((size_t)(v) * R + (s)) * RG_S]
#define HM_GOBJ(g) (obj0 + (long long)(g) * (VEC * RG_S))
  T* const chi = static_cast<T*>(P.chi);
  T* const Lm = static_cast<T*>(P.L);
  const T* const dat = static_cast<const T*>(P.data);

  copy_iter(&it, P.iter);
  if (tid < 2) cnt_sm[tid] = 0ull;
  if (!is_tail) {
    for (int g = 0; g < ngroups; ++g) {
      const long long base = HM_GOBJ(g);
      if (base >= obj_end) break;
      T tmp[VEC];
#pragma unroll
      for (int j = 0; j < p; ++j) {
        rg_load<T, VEC>(chi + j * Npad + base, tmp, false);
#pragma unroll
        for (int v = 0; v < VEC; ++v) HM_GAT(j, g * VEC + v) = tmp[v];
      }
#pragma unroll
      for (int k = 0; k < ntri; ++k) {
        rg_load<T, VEC>(Lm + k * Npad + base, tmp, false);
#pragma unroll
        for (int v = 0; v < VEC; ++v) HM_GAT(p + k, g * VEC + v) = tmp[v];
      }
#pragma unroll
      for (int c = 0; c < ncols; ++c) {
        rg_load<T, VEC>(dat + c * Npad + base, tmp, true);
#pragma unroll
        for (int v = 0; v < VEC; ++v) HM_GAT(p + ntri + c, g * VEC + v) = tmp[v];
      }
      DS ds;                                                   // draws of the launch's first iteration
      ds.make(P, base, (uint32_t)P.iter->t);
      ds.put(dr_my + (size_t)g * NV * RG_S, RG_S);
    }
  }
  __syncthreads();
  const long long t0 = it.t;

  if (!is_tail) {
    double nacc = 0.0, nnan = 0.0;
    for (long long k = 0; k < n_iter; ++k) {
      // the update starts as soon as the DECISION of iteration t - 1 is taken (theta_t's constants, eta, the moment count
      // are final then); theta'_t and its constants, which the tail warps are still deriving (~3,500 cycles), are needed only
      // by the population term at the end of the first object's update, which waits for them once (LateKp)
      if (k > 0) bar_sync(BAR_THETA, RG_THREADS);
      const SweepCtx<T> c = make_ctx<T>(P, it, t0 + k);
      int wait = k > 0 ? 1 : 0;
      const LateKp late{&it.kp, &wait, RG_THREADS};
      double acc[4] = {0.0, 0.0, 0.0, 0.0};
      for (int g = 0; g < ngroups; ++g) {
        // The one-off wait for theta' sits inside update_vec and is a block barrier: a warp must reach it CONVERGED.  So the
        // loop runs while ANY lane of the warp owns group g, and a lane that does not runs the update in lockstep on a
        // non-live dummy (base beyond N: nothing accumulated or stored; every access stays in its own shared-memory slots).
        const bool mine = HM_GOBJ(g) < obj_end;
        if (!__any_sync(0xffffffffu, mine)) break;
        const long long base = mine ? HM_GOBJ(g) : Npad + VEC;
        T x[p][VEC], l[ntri][VEC], d[ncols][VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
#pragma unroll
          for (int j = 0; j < p; ++j) x[j][v] = HM_GAT(j, g * VEC + v);
#pragma unroll
          for (int q = 0; q < ntri; ++q) l[q][v] = HM_GAT(p + q, g * VEC + v);
#pragma unroll
          for (int q = 0; q < ncols; ++q) d[q][v] = HM_GAT(p + ntri + q, g * VEC + v);
        }
        DS ds;
        ds.get(dr_my + (size_t)g * NV * RG_S, RG_S);
        update_vec<MODEL, T, false, false, true, VEC>(P, c, base, x, l, d, acc, &ds, &late);
        if (mine) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
#pragma unroll
          for (int j = 0; j < p; ++j) HM_GAT(j, g * VEC + v) = x[j][v];
#pragma unroll
          for (int q = 0; q < ntri; ++q) HM_GAT(p + q, g * VEC + v) = l[q][v];
        }
        }
      }
      if (wait) bar_sync(BAR_THETAP, RG_THREADS);             // a WARP without objects still takes part in the barrier (warp-uniform)
      nacc += acc[2]; nnan += acc[3];
      double v = acc[1];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
      if (lane == 0) red[k & 1][warp] = v;
      // (no fence needed: when the barrier completes, bar.arrive has ordered this thread's prior shared-memory writes for its participants)
      bar_arrive(BAR_PARTIALS, RG_THREADS);                   // hand the partials to the tail warps, do not wait
      if (k + 1 < n_iter) {                                   // the draws of iteration t + 1: overlaps the exchange and the theta step
        const uint32_t tn = (uint32_t)(t0 + k + 1);
        for (int g = 0; g < ngroups; ++g) {
          const long long base = HM_GOBJ(g);
          if (base >= obj_end) break;
          DS ds;
          ds.make(P, base, tn);
          ds.put(dr_my + (size_t)g * NV * RG_S, RG_S);
        }
      }
    }
    bar_sync(BAR_THETA, RG_THREADS);                          // the last tail has finished
    bar_sync(BAR_THETAP, RG_THREADS);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      nacc += __shfl_down_sync(0xffffffffu, nacc, o);
      nnan += __shfl_down_sync(0xffffffffu, nnan, o);
    }
    if (lane == 0) {
      atomicAdd(&cnt_sm[0], (unsigned long long)nacc);
      atomicAdd(&cnt_sm[1], (unsigned long long)nnan);
    }
    for (int g = 0; g < ngroups; ++g) {
      const long long base = HM_GOBJ(g);
      if (base >= obj_end) break;
      T tmp[VEC];
#pragma unroll
      for (int j = 0; j < p; ++j) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) tmp[v] = HM_GAT(j, g * VEC + v);
        rg_store<T, VEC>(chi + j * Npad + base, tmp);
      }
#pragma unroll
      for (int q = 0; q < ntri; ++q) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) tmp[v] = HM_GAT(p + q, g * VEC + v);
        rg_store<T, VEC>(Lm + q * Npad + base, tmp);
      }
    }
  } else {
    const int tw = warp - RG_SW, ttid = tid - RG_S;
    for (long long k = 0; k < n_iter; ++k) {
      bar_sync(BAR_PARTIALS, RG_THREADS);                     // the block's warp partials of iteration t0 + k
      double dq[1];
      dq[0] = lane < RG_SW ? red[k & 1][lane] : 0.0;
      lanes_to_total<1>(dq);
      unsigned long long* mb = P.mbox + (size_t)(k & 1) * mbox_parity_words(G);
      const unsigned epoch = epoch0 + (unsigned)k;
      mbox_push<1>(mb, G, (int)blockIdx.x, epoch, dq, ttid, RG_TW * 32);
      double tot[NPART] = {0.0, 0.0, 0.0, 0.0, 0.0};
      if (tw == 0) {
        double t1[1];
        mbox_collect<1>(mb + (size_t)blockIdx.x * mbox_reader_words(G), G, epoch, t1);
        tot[1] = t1[0];
      }
      tail_block<MODEL>(it, P.tail, tot, blockIdx.x == 0 ? P.trace : nullptr, tw, SyncNamed<BAR_TAIL, RG_TW * 32>(),
                        ArriveNamed<BAR_THETA, RG_THREADS>());   // theta_{t+1} is signalled after the decision phase ...
      // (no fence needed: when the barrier completes, bar.arrive has ordered this thread's prior shared-memory writes for its participants)
      bar_arrive(BAR_THETAP, RG_THREADS);                     // ... theta'_{t+1} and its constants when the tail is done
    }
  }
#undef HM_GAT
#undef HM_GOBJ
  __syncthreads();
  if (tid == 0) {
    P.blk_cnt[2 * blockIdx.x] += cnt_sm[0];
    P.blk_cnt[2 * blockIdx.x + 1] += cnt_sm[1];
  }
  if (blockIdx.x == 0) copy_iter(P.iter, &it);
}

}  // namespace hm
