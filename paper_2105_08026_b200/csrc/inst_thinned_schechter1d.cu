// inst_thinned_schechter1d.cu -- every kernel of model M_THINNED_SCHECHTER1D (its own translation unit: the models build in parallel).
// two Newton steps in log / sqrt (fastmath.cuh, HM_NEWTON_STEPS): measured faster for the on-chip p = 1 kernel of this model
#define HM_NEWTON_STEPS 2
#include "kernel_sets_impl.cuh"

namespace hm {

const void* kernel_sel_sweep_thinned_schechter1d();      // inst_thinned_schechter1d_selsweep.cu

bool kernels_thinned_schechter1d(int precision, int block, KernelSet* k, ResidentSet* r) {
  r->kernel = nullptr; r->kernel_sel_sweep = nullptr; r->n_base = 0; r->gen_kernel = nullptr; r->gen_kernel_v1 = nullptr; r->gen_values = 0; r->gen_vec = 0;
  if (precision == 0) {
    r->kernel = (const void*)k_resident<M_THINNED_SCHECHTER1D>; r->n_base = ResValues<M_THINNED_SCHECHTER1D>::n_base;
    r->kernel_sel_sweep = kernel_sel_sweep_thinned_schechter1d();
  }
  if (precision == 0) return pick_block<M_THINNED_SCHECHTER1D, double>(block, k);
  return false;
}

}  // namespace hm
