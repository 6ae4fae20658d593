// stream_tma.cuh -- HBM-streaming persistent Gibbs kernel with TMA-staged column loads (sm_100a).
// DESIGN.md section 8.6.
//
// Populations too large for shared memory (C3: 112 MB, C4: 280 MB per iteration) stream through the SMs every
// iteration.  In k_persistent (kernels.cuh) every warp alternates "issue 16-byte loads, wait ~1 us, compute",
// and with 16 resident warps per SM nothing hides that wait (ncu: 13 % long-scoreboard stalls, registers full of
// staged columns).  Here one elected thread per block streams the columns of the block's next tiles into a ring
// of shared-memory stages with bulk asynchronous copies (cp.async.bulk, the 1-D TMA path) that complete on an
// mbarrier; the 512 threads compute from shared memory and store chi and L straight from registers.
//   tile     = (blockDim.x - 32) * VEC consecutive objects: thread tid of block b owns, at step j, the VEC objects
//              starting at ((b + j G) (blockDim.x - 32) + tid) VEC -- a fixed map, so the reductions are
//              deterministic (the order differs from kernels.cuh::sweep, whose blocks have 32 more sweep threads)
//   stage    = the (p + ntri + ncols) columns of one tile, contiguous per column
//   pipeline = the block's tiles of an iteration in order, STAGES deep; the first tiles of iteration t+1 are
//              requested before the exchange and the theta tail of iteration t, so their latency overlaps them.
#pragma once
#include "kernels.cuh"
#include "resident_cfg.h"

namespace hm {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}
// global -> shared bulk copy, completion counted in bytes on `bar` (16-byte aligned addresses and size)
__device__ __forceinline__ void tma_load_1d(void* dst_smem, const void* src_gmem, unsigned bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}


// BLOCK threads = BLOCK - 32 consumers + one producer warp (a 17th warp would cost every thread a quarter of its
// registers: the register file is allocated per 4 warps).
template <int MODEL, class T, int BLOCK_ALL>
__global__ void __launch_bounds__(BLOCK_ALL, 1) k_persistent_tma(const Params P, const long long n_iter, const unsigned epoch0,
                                                                  const int n_stages) {
  constexpr int p = ModelDims<MODEL>::p, ntri = p * (p + 1) / 2, ncols = ModelDims<MODEL>::ncols;
  constexpr int BLOCK = BLOCK_ALL - 32;     // consumer threads
  constexpr int VEC = VecOf<T>::n, TILE = BLOCK * VEC, NC = p + ntri + ncols, NWC = BLOCK / 32;
  constexpr unsigned STAGE_BYTES = (unsigned)NC * TILE * sizeof(T);
  extern __shared__ __align__(128) unsigned char stage_mem[];
  __shared__ Iter it;
  __shared__ double red[32][NPART];
  __shared__ __align__(8) uint64_t full[TMA_MAX_STAGES], empty[TMA_MAX_STAGES];
  const int tid = (int)threadIdx.x, G = (int)gridDim.x, lane = tid & 31;
  const bool producer = tid >= BLOCK;
  const long long N = P.N, Npad = P.Npad;
  T* const chi = static_cast<T*>(P.chi);
  T* const Lm = static_cast<T*>(P.L);
  const T* const dat = static_cast<const T*>(P.data);
  const long long n_tiles = (N + TILE - 1) / TILE;
  const int my_tiles = blockIdx.x < n_tiles ? (int)((n_tiles - blockIdx.x + G - 1) / G) : 0;   // per iteration

  copy_iter(&it, P.iter);
  if (tid == 0) {
    for (int s = 0; s < n_stages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NWC); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // producer lane 0: request tile j (0-based within an iteration) of this block into the stage of pipeline slot q
  auto request = [&](const int j, const long long q) {
    const int s = (int)(q % n_stages);
    if (q >= n_stages) mbar_wait(&empty[s], (unsigned)((q / n_stages - 1) & 1));   // all consumer warps released it
    fence_proxy_async();
    const long long base = ((long long)blockIdx.x + (long long)j * G) * TILE;
    const long long n_el = Npad - base < TILE ? Npad - base : (long long)TILE;      // Npad is a multiple of 32 elements
    const unsigned col_bytes = (unsigned)(n_el * sizeof(T));
    unsigned char* dst = stage_mem + (size_t)s * STAGE_BYTES;
    mbar_expect_tx(&full[s], col_bytes * NC);
#pragma unroll
    for (int c = 0; c < NC; ++c) {
      const T* src = c < p ? chi + (long long)c * Npad + base
                           : (c < p + ntri ? Lm + (long long)(c - p) * Npad + base : dat + (long long)(c - p - ntri) * Npad + base);
      tma_load_1d(dst + (size_t)c * TILE * sizeof(T), src, col_bytes, &full[s]);
    }
  };

  long long q = 0;                       // pipeline slots of this block so far (same count in producer and consumers)
  const int n_pre = my_tiles < n_stages ? my_tiles : n_stages;
  if (producer && lane == 0) {
    for (int j = 0; j < n_pre; ++j) request(j, q + j);
  }
  double cnt[2] = {0.0, 0.0};
  for (long long k = 0; k < n_iter; ++k) {
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    double tq = 0.0;
    if (!producer) {
      const SweepCtx<T> c = make_ctx<T>(P, it);
      for (int j = 0; j < my_tiles; ++j) {
        const long long qq = q + j;
        const int s = (int)(qq % n_stages);
        mbar_wait(&full[s], (unsigned)((qq / n_stages) & 1));
        const T* st = reinterpret_cast<const T*>(stage_mem + (size_t)s * STAGE_BYTES) + VEC * tid;
        T x[p][VEC], l[ntri][VEC], d[ncols][VEC];
#pragma unroll
        for (int a = 0; a < p; ++a) ld_vec<T>(st + (size_t)a * TILE, x[a], false);
#pragma unroll
        for (int a = 0; a < ntri; ++a) ld_vec<T>(st + (size_t)(p + a) * TILE, l[a], false);
#pragma unroll
        for (int a = 0; a < ncols; ++a) ld_vec<T>(st + (size_t)(p + ntri + a) * TILE, d[a], false);
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);           // this warp holds its copy: the stage may be refilled
        const long long base = ((long long)blockIdx.x + (long long)j * G) * TILE + (long long)VEC * tid;
        if (base < N) {
          update_vec<MODEL, T, false>(P, c, base, x, l, d, acc);
#pragma unroll
          for (int a = 0; a < p; ++a) st_vec(chi + (long long)a * Npad + base, x[a]);
#pragma unroll
          for (int a = 0; a < ntri; ++a) st_vec(Lm + (long long)a * Npad + base, l[a]);
        }
      }
      tq = selection_slice<MODEL>(P, c.kp, BLOCK);
      __threadfence();                                   // this iteration's chi / L stores are at L2 ...
    } else if (lane == 0) {
      for (int j = n_pre; j < my_tiles; ++j) request(j, q + j);   // the rest of this iteration, as stages free up
    }
    q += my_tiles;
    cnt[0] += acc[2]; cnt[1] += acc[3];
    double dq[2] = {acc[1], tq};
    block_reduce_all<2>(dq, red);                        // ... (block barrier inside) ...
    if (producer && lane == 0 && k + 1 < n_iter) {       // ... before the async proxy re-reads them for iteration k+1:
      for (int j = 0; j < n_pre; ++j) request(j, q + j); //     requested now, they land during the exchange and the tail
    }
    constexpr int NVX = has_selection(MODEL) ? 2 : 1;   // only M1 / M4 have a selection-integral slice to exchange
    unsigned long long* mb = P.mbox + (size_t)(k & 1) * mbox_parity_words(G);
    const unsigned epoch = epoch0 + (unsigned)k;
    mbox_push<NVX>(mb, G, (int)blockIdx.x, epoch, dq, tid, BLOCK_ALL);
    double tot[NPART] = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (tid < 32) {
      double t2[2] = {0.0, 0.0};
      mbox_collect<NVX>(mb + (size_t)blockIdx.x * mbox_reader_words(G), G, epoch, t2);
      tot[1] = t2[0]; tot[2] = t2[1];
    }
    tail_block<MODEL>(it, P.tail, tot, blockIdx.x == 0 ? P.trace : nullptr, tid >> 5, SyncAll());
  }
  block_reduce_all<2>(cnt, red);
  if (tid == 0) {
    P.blk_cnt[2 * blockIdx.x] += (unsigned long long)cnt[0];
    P.blk_cnt[2 * blockIdx.x + 1] += (unsigned long long)cnt[1];
  }
  if (blockIdx.x == 0) copy_iter(P.iter, &it);
}

}  // namespace hm
