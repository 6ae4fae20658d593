// resident.cuh -- the on-chip variant of the persistent Gibbs kernel for populations that fit in shared memory
// (fp64, p = 1: BASELINE configs C0, C1, C2).  DESIGN.md section 8.5.
//
// At N = 3e5 an iteration moves 24 MB (3.7 us at HBM peak) and the exchange + theta tail is a serial chain of
// ~4 us that no amount of bandwidth shortens (profiles/r01b).  This kernel removes both from the critical path:
//   - every object lives in the shared memory of the block that owns it for the whole launch (chi, L, data,
//     moments, e^chi): HBM/L2 are touched at launch start and end only;
//   - the sweep is split into a theta-INDEPENDENT front (Philox draws, Box-Muller, chi' = chi + L z, e^chi') and
//     a theta-dependent back (log targets, accept, RAM update, population terms, moments).  Sweep warps run
//     back(t) -> hand their partials to the tail warps -> front(t+1) while 4 dedicated tail warps do the
//     grid-wide exchange and the theta step of iteration t; the sweep warps only wait for theta_{t+1} if the
//     tail is still running when their front is done.
// Same arithmetic per object as kernels.cuh::sweep (same Plate<> functors, same draws); only the order in which
// block partials are added differs (fixed, so still deterministic).
#pragma once
#include "kernels.cuh"
#include "resident_cfg.h"

namespace hm {

#ifndef HM_RES_IL
#define HM_RES_IL 2
#endif
constexpr int RES_IL = HM_RES_IL;                   // slots of the back processed together (instruction-level parallelism)

// per-object values kept in shared memory: [value][slot r][sweep thread]
template <int MODEL> struct ResValues {
  static constexpr int ncols = ModelDims<MODEL>::ncols;
  static constexpr bool m1 = has_selection(MODEL);     // M1 / M4: e^chi cached next to chi, selection sum on the tail warps
  static constexpr int V_CHI = 0, V_L = 1, V_D = 2, V_XP = 2 + ncols, V_U = 3 + ncols, V_E = 4 + ncols, V_EP = 5 + ncols;
  static constexpr int n_base = 4 + ncols + (m1 ? 2 : 0);   // + 2 (mean, M2) when moments are kept
};

// 8-byte asynchronous copy global -> shared (LDGSTS); completion per thread with cp_async_wait_all
__device__ __forceinline__ void cp_async8(double* dst_smem, const double* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }


// SEL_SWEEP (M1 with few slots per thread, e.g. C1): the selection sum at theta' is computed by the 512 SWEEP threads, two
// nodes each, right after theta' arrives, and handed to the tail warps with the Delta partials -- instead of by the 128 tail
// threads after the theta tail, where a short sweep leaves it on the critical path (C1: 4.80 -> 4.5 us per iteration).  A
// variant of its own because the default kernel's code generation must not move (C2 loses 0.1 us to a run-time switch), and
// not used for M4, whose node term (exp and expm1) is long enough to cost the sweep warps more than it saves the tail.
template <int MODEL, bool SEL_SWEEP = false>
__global__ void __launch_bounds__(RES_THREADS, 1) k_resident(const Params P, const long long n_iter, const unsigned epoch0,
                                                             const int R, const int OB) {
  using T = double;
  using V = ResValues<MODEL>;
  using PL = Plate<MODEL, T>;
  constexpr int ncols = V::ncols;
  extern __shared__ double sm[];
  __shared__ Iter it;
  __shared__ double red[2][RES_SW][SEL_SWEEP ? 2 : 1];   // per sweep warp: Delta partial (and selection-sum partial)
  __shared__ unsigned long long cnt_sm[2];
  __shared__ double qtab[V::m1 ? 3 : 1][V::m1 ? NQUAD : 1];   // M1: quadrature weights W_k, nodes x_k, e^{x_k}
  __shared__ double tq_warp[RES_TW];     // M1: the tail warps' partial sums of the selection integral at theta'
  const int tid = (int)threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const bool is_tail = warp >= RES_SW;
  const int G = (int)gridDim.x;
  const long long N = P.N, Npad = P.Npad;
  const bool keep_mom = P.tail.keep_moments != 0;
  const int V_MEAN = V::n_base, V_M2 = V::n_base + 1;
  // A block owns the OB (even) contiguous objects [blockIdx.x * OB, (blockIdx.x + 1) * OB), so the population is
  // spread evenly over the grid; a thread owns adjacent PAIRS of them (objects draw in pairs,
  // kernels.cuh::pair_draws): slot r = 2a + h is object obj0 + 2 a RES_S + h.  R = 2 ceil(OB / (2 RES_S)).
  const long long obj0 = (long long)blockIdx.x * OB + 2 * tid;
  const long long obj_end = (long long)(blockIdx.x + 1) * OB < N ? (long long)(blockIdx.x + 1) * OB : N;
#define HM_OBJ(r) (obj0 + (long long)((r) >> 1) * (2 * RES_S) + ((r) & 1))
  int nlive = 0;                                                  // HM_OBJ increases with r: live slots are 0 .. nlive-1
  for (int r = 0; r < R; ++r) nlive += HM_OBJ(r) < obj_end ? 1 : 0;
  T* const chi = static_cast<T*>(P.chi);
  T* const Lm = static_cast<T*>(P.L);
  const T* const dat = static_cast<const T*>(P.data);
  double* const my = sm + tid;
#define HM_AT(v, r) my[((v) * R + (r)) * RES_S]

  copy_iter(&it, P.iter);
  if (tid < 2) cnt_sm[tid] = 0ull;
  if constexpr (SEL_SWEEP) {
    static_assert(!SEL_SWEEP || V::m1, "SEL_SWEEP is for the models with a selection sum");
    for (int q = tid; q < NQUAD; q += RES_THREADS) { qtab[0][q] = P.qW[q]; qtab[1][q] = P.qx[q]; qtab[2][q] = P.qex[q]; }
  }
  if (!is_tail) {
    // The state comes on chip with asynchronous 8-byte copies (cp.async: global -> shared without passing through
    // registers; a thread's slot pair is two adjacent objects, so a warp still reads whole 512-byte runs per column) ...
    for (int r = 0; r < nlive; ++r) {
      const long long i = HM_OBJ(r);
      cp_async8(&HM_AT(V::V_CHI, r), chi + i);
      cp_async8(&HM_AT(V::V_L, r), Lm + i);
#pragma unroll
      for (int c = 0; c < ncols; ++c) cp_async8(&HM_AT(V::V_D + c, r), dat + c * Npad + i);
      if (keep_mom) { cp_async8(&HM_AT(V_MEAN, r), P.mom_mean + i); cp_async8(&HM_AT(V_M2, r), P.mom_M2 + i); }
    }
    cp_async_commit();
    // ... and while they are in flight the thread makes the plate draws of the launch's first front, which depend on
    // (seed, object, t) only (the normal is parked in the chi' slot)
    const uint32_t t_first = (uint32_t)P.iter->t;
    for (int r = 0; r < nlive; r += 2) {
      T z[2][2], cs[2], sn[2], u[2];
      pair_draws<1, 2>((uint64_t)P.tail.seed, P.obj_offset + HM_OBJ(r), t_first, z, cs, sn, u);
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        if (r + h < nlive) { HM_AT(V::V_XP, r + h) = z[h][0]; HM_AT(V::V_U, r + h) = u[h]; }
      }
    }
    cp_async_wait_all();
    for (int r = 0; r < nlive; ++r) {                        // the rest of the first front: chi' = chi + L z, e^chi, e^chi'
      const T x = HM_AT(V::V_CHI, r);
      const T xp = x + HM_AT(V::V_L, r) * HM_AT(V::V_XP, r);
      HM_AT(V::V_XP, r) = xp;
      if (V::m1) { HM_AT(V::V_E, r) = hm_exp(x); HM_AT(V::V_EP, r) = hm_exp_point(xp); }
    }
  }
  __syncthreads();
  const long long t0 = it.t;

  if (!is_tail) {
    // theta-independent half of the update of iteration t: pair draws, proposals, e^chi'
    auto front = [&](const uint32_t t) {
      for (int r = 0; r < nlive; r += 2) {
        T z[2][2], cs[2], sn[2], u[2];
        pair_draws<1, 2>((uint64_t)P.tail.seed, P.obj_offset + HM_OBJ(r), t, z, cs, sn, u);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          if (r + h < nlive) {
            const T xp = HM_AT(V::V_CHI, r + h) + HM_AT(V::V_L, r + h) * z[h][0];
            HM_AT(V::V_XP, r + h) = xp;
            HM_AT(V::V_U, r + h) = u[h];
            if (V::m1) HM_AT(V::V_EP, r + h) = hm_exp_point(xp);
          }
        }
      }
    };
    T mcT[MC_N];
#pragma unroll
    for (int j = 0; j < MC_N; ++j) mcT[j] = (T)P.mc[j];
    const T astar = (T)P.astar_chi;
    double nacc = 0.0, nnan = 0.0;

    for (long long k = 0; k < n_iter; ++k) {
      const long long t = t0 + k;
      if (k > 0) bar_sync(BAR_THETA, RES_THREADS);          // theta_t and everything derived from it are in `it`
      // back, part 1 (needs theta_t only): targets, accept, RAM update, new chi, moments
      const ThetaK kc = it.kc;
      const KT<T> kT = narrow<T>(kc);
      const T eta = (T)it.dr[slot3(t)].eta;
      const bool do_mom = keep_mom && t > P.tail.burn_in;
      const double inv_k = it.inv_k;
      // RES_IL slots at a time in straight-line code: the back sits on the critical path of the iteration (the
      // exchange cannot start before it ends) and one slot is a single dependent chain of fp64 operations, so with
      // 4 warps per scheduler it is latency-bound; independent slots interleave.  A slot past nlive repeats the
      // last live one and is not stored.
      for (int r = 0; r < nlive; r += RES_IL) {
        T xi[RES_IL], yi[RES_IL], la[RES_IL], lnew[RES_IL], exq[RES_IL];
        bool acc[RES_IL], bad[RES_IL];
        int rr[RES_IL];
#pragma unroll
        for (int j = 0; j < RES_IL; ++j) {
          rr[j] = r + j < nlive ? r + j : nlive - 1;
          T di[ncols];
#pragma unroll
          for (int c = 0; c < ncols; ++c) di[c] = HM_AT(V::V_D + c, rr[j]);
          xi[j] = HM_AT(V::V_CHI, rr[j]); yi[j] = HM_AT(V::V_XP, rr[j]);
          typename PL::Pt qc, qp;
          if constexpr (V::m1) {
            qc = typename PL::Pt{xi[j], HM_AT(V::V_E, rr[j])};
            qp = typename PL::Pt{yi[j], HM_AT(V::V_EP, rr[j])};
            exq[j] = qp.ex;
          } else {
            qc = PL::point(&xi[j]); qp = PL::point(&yi[j]);
            exq[j] = T(0);
          }
          const T pc = PL::target(qc, di, kT, mcT), pp = PL::target(qp, di, kT, mcT);
          const T diff = pp - pc;
          bad[j] = diff != diff;
          la[j] = bad[j] ? T(-INFINITY) : (diff < T(0) ? diff : T(0));
        }
#pragma unroll
        for (int j = 0; j < RES_IL; ++j) {
          const T alpha = hm_exp_nonpos(la[j]);
          acc[j] = HM_AT(V::V_U, rr[j]) < alpha;
          lnew[j] = HM_AT(V::V_L, rr[j]) * hm_sqrt_pos(T(1) + eta * (alpha - astar));
        }
#pragma unroll
        for (int j = 0; j < RES_IL; ++j) {
          if (r + j < nlive) {
            nacc += acc[j] ? 1.0 : 0.0; nnan += bad[j] ? 1.0 : 0.0;
            HM_AT(V::V_L, rr[j]) = lnew[j];
            if (acc[j]) {
              HM_AT(V::V_CHI, rr[j]) = yi[j];
              if constexpr (V::m1) HM_AT(V::V_E, rr[j]) = exq[j];
            }
            if (do_mom) {
              const double xv = (double)(acc[j] ? yi[j] : xi[j]), m0 = HM_AT(V_MEAN, rr[j]);
              const double dl = xv - m0, m1 = m0 + dl * inv_k;
              HM_AT(V_MEAN, rr[j]) = m1;
              HM_AT(V_M2, rr[j]) += dl * (xv - m1);
            }
          }
        }
      }
      // back, part 2 (needs theta'_t, which the tail finishes a little later): population terms.  (M1's selection
      // integral at theta' is computed by the tail warps, see below: every value less in the exchange is worth more
      // than the arithmetic it saves -- a third mailbox value measured +0.7 us per iteration.)
      if (k > 0) bar_sync(BAR_THETAP, RES_THREADS);
      const ThetaK kp = it.kp;
      double v[2] = {0.0, 0.0};
      for (int r = 0; r < nlive; ++r) {
        T di[ncols];
#pragma unroll
        for (int c = 0; c < ncols; ++c) di[c] = HM_AT(V::V_D + c, r);
        const T xn = HM_AT(V::V_CHI, r);
        typename PL::Pt qn;
        if constexpr (V::m1) qn = typename PL::Pt{xn, HM_AT(V::V_E, r)}; else qn = PL::point(&xn);
        v[0] += PL::pop(qn, di, kp, P.mc) - PL::pop(qn, di, kc, P.mc);
      }
      if constexpr (SEL_SWEEP) {
        static_assert(NQUAD % RES_S == 0, "quadrature nodes must divide over the sweep threads");
        if (!P.tail.freeze_theta) {
#pragma unroll
          for (int m = 0; m < NQUAD / RES_S; ++m) {
            const int q = tid + m * RES_S;
            v[1] += selection_term<MODEL>(kp, qtab[0][q], qtab[1][q], qtab[2][q]);
          }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[1] += __shfl_down_sync(0xffffffffu, v[1], o);
        if (lane == 0) red[k & 1][warp][SEL_SWEEP ? 1 : 0] = v[1];
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v[0] += __shfl_down_sync(0xffffffffu, v[0], o);
      if (lane == 0) red[k & 1][warp][0] = v[0];
      // (no fence needed: when the barrier completes, bar.arrive has ordered this thread's prior shared-memory writes for its participants)
      bar_arrive(BAR_PARTIALS, RES_THREADS);                 // hand the partials to the tail warps, do not wait
      if (k + 1 < n_iter) front((uint32_t)(t + 1));          // overlaps the exchange and the theta step
    }
    bar_sync(BAR_THETA, RES_THREADS);                        // the last tail has finished
    bar_sync(BAR_THETAP, RES_THREADS);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      nacc += __shfl_down_sync(0xffffffffu, nacc, o);
      nnan += __shfl_down_sync(0xffffffffu, nnan, o);
    }
    if (lane == 0) {
      atomicAdd(&cnt_sm[0], (unsigned long long)nacc);
      atomicAdd(&cnt_sm[1], (unsigned long long)nnan);
    }
    for (int r = 0; r < nlive; r += 2) {
      const long long i = HM_OBJ(r);
      if (r + 1 < nlive) {
        *reinterpret_cast<double2*>(chi + i) = make_double2(HM_AT(V::V_CHI, r), HM_AT(V::V_CHI, r + 1));
        *reinterpret_cast<double2*>(Lm + i) = make_double2(HM_AT(V::V_L, r), HM_AT(V::V_L, r + 1));
        if (keep_mom) {
          *reinterpret_cast<double2*>(P.mom_mean + i) = make_double2(HM_AT(V_MEAN, r), HM_AT(V_MEAN, r + 1));
          *reinterpret_cast<double2*>(P.mom_M2 + i) = make_double2(HM_AT(V_M2, r), HM_AT(V_M2, r + 1));
        }
      } else {
        chi[i] = HM_AT(V::V_CHI, r);
        Lm[i] = HM_AT(V::V_L, r);
        if (keep_mom) { P.mom_mean[i] = HM_AT(V_MEAN, r); P.mom_M2[i] = HM_AT(V_M2, r); }
      }
    }
  } else {
    const int tw = warp - RES_SW, ttid = tid - RES_S;
    // M1: T(theta') needs sum_k W_k phi(x_k; theta') over the 1,024 quadrature nodes.  Every block computes the
    // whole sum itself on its tail warps right after theta' is known -- while the sweep warps are busy with the
    // next back -- in a fixed order: all blocks hold the same bits and only ONE value per block (Delta) has to be
    // exchanged.  Node tables in shared memory (24 KB), loaded once per launch.
    constexpr int QPT = NQUAD / (RES_TW * 32);
    static_assert(NQUAD % (RES_TW * 32) == 0, "quadrature nodes must divide over the tail threads");
    if constexpr (V::m1 && !SEL_SWEEP) {
      for (int q = ttid; q < NQUAD; q += RES_TW * 32) { qtab[0][q] = P.qW[q]; qtab[1][q] = P.qx[q]; qtab[2][q] = P.qex[q]; }
    }
    auto selection_full = [&]() {
      if constexpr (V::m1) {
        if (!P.tail.freeze_theta) {
          const ThetaK kq = it.kp;
          double s_ = 0.0;
#pragma unroll
          for (int m = 0; m < QPT; ++m) {
            const int q = ttid + m * RES_TW * 32;
            s_ += selection_term<MODEL>(kq, qtab[0][q], qtab[1][q], qtab[2][q]);
          }
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) s_ += __shfl_down_sync(0xffffffffu, s_, o);
          if (lane == 0) tq_warp[tw] = s_;
        }
        bar_sync(BAR_TAIL, RES_TW * 32);
      }
    };
    if constexpr (!SEL_SWEEP) selection_full();
    for (long long k = 0; k < n_iter; ++k) {
      bar_sync(BAR_PARTIALS, RES_THREADS);                   // the block's 16 warp partials of iteration t0 + k
      double dq[1];
      dq[0] = lane < RES_SW ? red[k & 1][lane][0] : 0.0;
      lanes_to_total<1>(dq);
      double tq[1] = {0.0};
      if constexpr (SEL_SWEEP) {                             // the sweep warps' partials of the selection sum, same fixed order
        tq[0] = lane < RES_SW ? red[k & 1][lane][SEL_SWEEP ? 1 : 0] : 0.0;
        lanes_to_total<1>(tq);
      }
      unsigned long long* mb = P.mbox + (size_t)(k & 1) * mbox_parity_words(G);
      const unsigned epoch = epoch0 + (unsigned)k;
      mbox_push<1>(mb, G, (int)blockIdx.x, epoch, dq, ttid, RES_TW * 32);
      double tot[NPART] = {0.0, 0.0, 0.0, 0.0, 0.0};
      if (tw == 0) {
        double t1[1];
        mbox_collect<1>(mb + (size_t)blockIdx.x * mbox_reader_words(G), G, epoch, t1);
        tot[1] = t1[0];
        if constexpr (SEL_SWEEP) tot[2] = tq[0];
        else if constexpr (V::m1) tot[2] = ((tq_warp[0] + tq_warp[1]) + tq_warp[2]) + tq_warp[3];
      }
      tail_block<MODEL>(it, P.tail, tot, blockIdx.x == 0 ? P.trace : nullptr, tw, SyncNamed<BAR_TAIL, RES_TW * 32>(),
                 ArriveNamed<BAR_THETA, RES_THREADS>());      // theta_{t+1} is signalled after the decision phase ...
      // (no fence needed: when the barrier completes, bar.arrive has ordered this thread's prior shared-memory writes for its participants)
      bar_arrive(BAR_THETAP, RES_THREADS);                   // ... theta'_{t+1} and its constants when the tail is done
      if constexpr (!SEL_SWEEP) selection_full();            // M1: for the NEXT decision; off the critical path
    }
  }
#undef HM_AT
#undef HM_OBJ
  __syncthreads();
  if (tid == 0) {
    P.blk_cnt[2 * blockIdx.x] += cnt_sm[0];
    P.blk_cnt[2 * blockIdx.x + 1] += cnt_sm[1];
  }
  if (blockIdx.x == 0) copy_iter(P.iter, &it);
}

}  // namespace hm
