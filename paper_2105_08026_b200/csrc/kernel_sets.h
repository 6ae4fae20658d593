// kernel_sets.h -- the table of kernel entry points of one (model, precision, block size), filled by the per-model
// translation units inst_*.cu (one per compiled-in model, so that they build in parallel) and read by cudahm.cu.
#pragma once
#include <cstddef>

namespace hm {

struct KernelSet {
  const void* persistent;          // plain streaming persistent kernel
  const void* persistent_ahead;    // the variant with staged draws / L2 prefetch
  size_t stage_step_bytes;         // shared memory of one staged step of plate draws (DrawSet::NV x BLOCK values)
  const void* persistent_tma;
  size_t tma_stage_bytes;
  const void* sweep;
  const void* sweep_tap;
  const void* init_state;
  // the frozen-member variants (update mask / per-object counter)
  const void* persistent_hold;
  const void* sweep_hold;
  const void* sweep_tap_hold;
  // streaming kernel with dedicated tail warps (k_persistent_dt) and its sweep threads per block; NULL where not built
  const void* persistent_dt;
  const void* persistent_dt_nomom;   // ... compiled without the running-moments update (handles with keep_chi_moments = 0)
  int dt_sweep_threads;
  const void* sweep_dt;          // k_sweep / tapped k_sweep at the same thread -> object map
  const void* sweep_tap_dt;
};

// on-chip kernel (resident.cuh) of one (model, precision)
struct ResidentSet {
  const void* kernel;              // NULL: the model has no on-chip kernel in this precision
  int n_base;                      // shared-memory values per object without the running moments (+ 2 with them)
  const void* kernel_sel_sweep;    // variant whose sweep warps compute the selection sum (few slots per thread); may be NULL
  // the general on-chip kernel (resident_gen.cuh; p >= 2, fp32 state): entry point, values of T per object, objects per
  // thread group (16 bytes of T)
  const void* gen_kernel;
  int gen_values, gen_vec;
  const void* gen_kernel_v1;       // the same kernel with ONE object per thread (fp64, p >= 2; small populations); may be NULL
};

// each returns false when the (precision, block) combination is not compiled in for that model
bool kernels_normal1d(int precision, int block, KernelSet* k, ResidentSet* r);
bool kernels_thinned_schechter1d(int precision, int block, KernelSet* k, ResidentSet* r);
bool kernels_binormal2d(int precision, int block, KernelSet* k, ResidentSet* r);
bool kernels_linreg_me1d(int precision, int block, KernelSet* k, ResidentSet* r);
bool kernels_bb1_fluxnoise1d(int precision, int block, KernelSet* k, ResidentSet* r);
bool kernels_normal3d_knowncov(int precision, int block, KernelSet* k, ResidentSet* r);
bool kernels_normal4d_knowncov(int precision, int block, KernelSet* k, ResidentSet* r);   // p >= 4: 256-thread blocks only
bool kernels_normal5d_knowncov(int precision, int block, KernelSet* k, ResidentSet* r);
bool kernels_normal6d_knowncov(int precision, int block, KernelSet* k, ResidentSet* r);

}  // namespace hm
