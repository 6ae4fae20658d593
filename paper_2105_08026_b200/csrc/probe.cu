// probe.cu -- launch / sync / barrier floors and ALU-pipe peaks (include/cudahm_probe.h).
#include "cudahm_probe.h"
#include "fastmath.cuh"

#include <cuda_runtime.h>
#include <vector>

namespace {

__global__ void k_empty(int* sink) { if (sink && threadIdx.x == 0xffffffffu) *sink = 1; }

// same barrier as kernels.cuh::grid_barrier (kept textually separate so the probe cannot perturb the sampler)
__global__ void k_barrier_loop(unsigned* bar, int n) {
  const unsigned G = gridDim.x;
  for (int k = 0; k < n; ++k) {
    __syncthreads();
    if (threadIdx.x == 0) {
      asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
      unsigned v;
      const unsigned target = (unsigned)(k + 1) * G;
      do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory"); } while (v < target);
    }
    __syncthreads();
  }
}

template <class T>
__global__ void k_fma(T* out, int iters) {
  T a[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) a[j] = (T)(threadIdx.x + j) * (T)1e-3;
  const T m = (T)0.999999, c = (T)1e-7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int j = 0; j < 8; ++j) a[j] = a[j] * m + c;
    }
  }
  T s = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) s += a[j];
  if (s == (T)123456789) out[0] = s;
}

#define PR_TRY(call) do { if ((call) != cudaSuccess) { cudaGetLastError(); rc = -3; goto done; } } while (0)

}  // namespace

extern "C" int cudahm_probe_floor(void* cuda_stream, int kind, int n_iter, int grid_blocks, int block_threads,
                                  double* us_per_iter) {
  if (!us_per_iter || n_iter < 1 || kind < 0 || kind > 3) return -1;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0, rc = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -3;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int grid = grid_blocks > 0 ? grid_blocks : sms, block = block_threads > 0 ? block_threads : 512;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  unsigned* bar = nullptr; double* hbuf = nullptr; cudaGraph_t g = nullptr; cudaGraphExec_t ge = nullptr;
  cudaStream_t cap = nullptr;
  float ms = 0.f;
  int* null_sink = nullptr;
  PR_TRY(cudaEventCreate(&e0)); PR_TRY(cudaEventCreate(&e1));
  PR_TRY(cudaMalloc((void**)&bar, 256)); PR_TRY(cudaHostAlloc((void**)&hbuf, 64, cudaHostAllocDefault));
  for (int rep = 0; rep < 2; ++rep) {     // rep 0 = warm-up
    PR_TRY(cudaMemsetAsync(bar, 0, 4, st));
    if (kind == CUDAHM_FLOOR_GRAPH && !ge) {
      PR_TRY(cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
      PR_TRY(cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal));
      for (int k = 0; k < 50; ++k) { k_empty<<<grid, block, 0, cap>>>(null_sink); k_empty<<<1, 32, 0, cap>>>(null_sink); }
      PR_TRY(cudaStreamEndCapture(cap, &g));
      PR_TRY(cudaGraphInstantiate(&ge, g, 0));
    }
    PR_TRY(cudaEventRecord(e0, st));
    if (kind == CUDAHM_FLOOR_LAUNCH) {
      for (int k = 0; k < n_iter; ++k) { k_empty<<<grid, block, 0, st>>>(null_sink); k_empty<<<1, 32, 0, st>>>(null_sink); }
    } else if (kind == CUDAHM_FLOOR_GRAPH) {
      for (int k = 0; k < (n_iter + 49) / 50; ++k) PR_TRY(cudaGraphLaunch(ge, st));
    } else if (kind == CUDAHM_FLOOR_GRID_BARRIER) {
      int n = n_iter;
      void* args[] = {&bar, &n};
      PR_TRY(cudaLaunchCooperativeKernel((const void*)k_barrier_loop, dim3(grid), dim3(block), args, 0, st));
    } else {
      for (int k = 0; k < n_iter; ++k) {
        k_empty<<<grid, block, 0, st>>>(null_sink); k_empty<<<1, 32, 0, st>>>(null_sink);
        PR_TRY(cudaMemcpyAsync(hbuf, bar, 40, cudaMemcpyDeviceToHost, st));
        PR_TRY(cudaStreamSynchronize(st));
      }
    }
    PR_TRY(cudaEventRecord(e1, st));
    PR_TRY(cudaStreamSynchronize(st));
    PR_TRY(cudaGetLastError());
    PR_TRY(cudaEventElapsedTime(&ms, e0, e1));
  }
  {
    const int done_iters = kind == CUDAHM_FLOOR_GRAPH ? (n_iter + 49) / 50 * 50 : n_iter;
    *us_per_iter = 1e3 * (double)ms / done_iters;
  }
done:
  if (ge) cudaGraphExecDestroy(ge);
  if (g) cudaGraphDestroy(g);
  if (cap) cudaStreamDestroy(cap);
  if (bar) cudaFree(bar);
  if (hbuf) cudaFreeHost(hbuf);
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  return rc;
}

extern "C" int cudahm_probe_fma_peak(void* cuda_stream, int dtype, double* tera_fma_per_s) {
  if (!tera_fma_per_s || dtype < 0 || dtype > 1) return -1;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0, rc = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -3;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int grid = sms * 4, block = 512, iters = 4096;
  cudaEvent_t e0 = nullptr, e1 = nullptr; void* out = nullptr; float ms = 0.f, best = 1e30f;
  PR_TRY(cudaEventCreate(&e0)); PR_TRY(cudaEventCreate(&e1)); PR_TRY(cudaMalloc(&out, 64));
  for (int rep = 0; rep < 4; ++rep) {
    PR_TRY(cudaEventRecord(e0, st));
    if (dtype == 0) k_fma<double><<<grid, block, 0, st>>>((double*)out, iters);
    else k_fma<float><<<grid, block, 0, st>>>((float*)out, iters);
    PR_TRY(cudaEventRecord(e1, st));
    PR_TRY(cudaStreamSynchronize(st));
    PR_TRY(cudaGetLastError());
    PR_TRY(cudaEventElapsedTime(&ms, e0, e1));
    if (rep > 0 && ms < best) best = ms;
  }
  *tera_fma_per_s = (double)grid * block * (double)iters * 64.0 / ((double)best * 1e-3) * 1e-12;
done:
  if (out) cudaFree(out);
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  return rc;
}

namespace {
__global__ void k_probe_math(const int fn, const double* __restrict__ x, double* __restrict__ y, const long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double v = x[i];
  double r = 0.0, q = 0.0;
  switch (fn) {
    case CUDAHM_MATH_EXP: r = hm::hm_exp_fast(v); break;
    case CUDAHM_MATH_EXPM1_NONPOS: r = hm::hm_expm1_nonpos(v); break;
    case CUDAHM_MATH_LOG: r = hm::hm_log_pos_n<1>(v); break;
    case CUDAHM_MATH_SQRT: r = hm::hm_sqrt_fast_n<1>(v); break;
    case CUDAHM_MATH_SQRT_BOTH_ROOT: hm::hm_sqrt_rsqrt_n<1>(v, &r, &q); break;
    case CUDAHM_MATH_SQRT_BOTH_INV: hm::hm_sqrt_rsqrt_n<1>(v, &q, &r); break;
    case CUDAHM_MATH_LOG_2: r = hm::hm_log_pos_n<2>(v); break;
    case CUDAHM_MATH_SQRT_2: r = hm::hm_sqrt_fast_n<2>(v); break;
    case CUDAHM_MATH_SQRT_BOTH_ROOT_2: hm::hm_sqrt_rsqrt_n<2>(v, &r, &q); break;
    case CUDAHM_MATH_SQRT_BOTH_INV_2: hm::hm_sqrt_rsqrt_n<2>(v, &q, &r); break;
    case CUDAHM_MATH_SIN2PI: hm::hm_sincos2pi(v, &r, &q); break;
    default: hm::hm_sincos2pi(v, &q, &r); break;
  }
  y[i] = r;
}
}  // namespace

extern "C" int cudahm_probe_math(void* cuda_stream, int fn, const double* x_host, double* y_host, long long n) {
  if (!x_host || !y_host || n < 0 || fn < CUDAHM_MATH_EXP || fn > CUDAHM_MATH_SQRT_BOTH_INV_2) return -1;
  if (n == 0) return 0;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = 0;
  double *x = nullptr, *y = nullptr;
  PR_TRY(cudaMalloc(&x, (size_t)n * 8)); PR_TRY(cudaMalloc(&y, (size_t)n * 8));
  PR_TRY(cudaMemcpyAsync(x, x_host, (size_t)n * 8, cudaMemcpyHostToDevice, st));
  k_probe_math<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(fn, x, y, n);
  PR_TRY(cudaGetLastError());
  PR_TRY(cudaMemcpyAsync(y_host, y, (size_t)n * 8, cudaMemcpyDeviceToHost, st));
  PR_TRY(cudaStreamSynchronize(st));
done:
  if (x) cudaFree(x);
  if (y) cudaFree(y);
  return rc;
}
