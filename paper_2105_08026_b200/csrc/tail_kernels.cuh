// tail_kernels.cuh -- the non-template kernels (theta tail as its own launch, iteration set-up, moment read-out).
// Included by cudahm.cu only (the per-model translation units inst_*.cu hold the templates of kernels.cuh).
#pragma once
#include "kernels.cuh"

namespace hm {

// Tail kernel: reduce the slots (TAIL_REDUCE: also publish the totals for the host); TAIL_DECIDE: the
// block-parallel theta tail, which decides iteration t and prepares t + 1.
enum : int { TAIL_REDUCE = 1, TAIL_DECIDE = 2 };
constexpr int TAIL_THREADS = 128;
__global__ void __launch_bounds__(TAIL_THREADS, 1) k_tail(const Params P, const int nblocks, const int flags) {
  __shared__ Iter it;
  copy_iter(&it, P.iter);
  __syncthreads();
  double tot[NPART] = {0.0, 0.0, 0.0, 0.0, 0.0};
  if (threadIdx.x < 32) {
    slots_reduce(P.slots, nblocks, tot);
    if ((flags & TAIL_REDUCE) && threadIdx.x == 0) {
#pragma unroll
      for (int q = 0; q < NPART; ++q) P.totals[q] = tot[q];
    }
  }
  if (flags & TAIL_DECIDE) {
    tail_block(it, P.tail, tot, P.trace, (int)(threadIdx.x >> 5), SyncAll());
    __syncthreads();
    copy_iter(P.iter, &it);
  }
}

// After set_init / set_state: derive kc, log prior and T(theta) for the uploaded theta, then prepare it.t.
__global__ void __launch_bounds__(256, 1) k_init_iter(const Params P) {
  __shared__ Iter it;
  __shared__ double red[32][NPART];
  copy_iter(&it, P.iter);
  __syncthreads();
  const ThetaK kc = theta_consts(P.tail.model, it.theta);
  double part[NPART] = {0, 0, 0, 0, 0};
  if (has_selection(P.tail.model)) {
    for (int k = threadIdx.x; k < NQUAD; k += blockDim.x)
      part[2] += selection_term_rt(P.tail.model, kc, P.qW[k], P.qx[k], P.qex[k]);
  }
  block_reduce<NPART>(part, red);
  if (threadIdx.x == 0) {
    it.kc = kc;
    it.lp_cur = log_prior_full(P.tail, it.theta);
    it.T_cur = has_selection(P.tail.model) ? theta_only_from_sum(P.tail.model, kc, part[2], P.tail.n_objects) : 0.0;
    prepare_iteration(it, P.tail, it.t);
  }
  __syncthreads();
  copy_iter(P.iter, &it);
}

__global__ void k_fill_u32(unsigned* v, long long n, unsigned value) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) v[i] = value;
}

// sample variance from the Welford sums, written next to them for read-out
__global__ void k_finalize_moments(const double* M2, double* var, long long n, double inv_km1) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) var[i] = M2[i] * inv_km1;
}

}  // namespace hm
