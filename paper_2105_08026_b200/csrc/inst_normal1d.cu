// inst_normal1d.cu -- every kernel of model M_NORMAL1D (its own translation unit: the models build in parallel).
// two Newton steps in log / sqrt (fastmath.cuh, HM_NEWTON_STEPS): measured faster for the on-chip p = 1 kernel of this model
#define HM_NEWTON_STEPS 2
#include "kernel_sets_impl.cuh"

namespace hm {

bool kernels_normal1d(int precision, int block, KernelSet* k, ResidentSet* r) {
  r->kernel = nullptr; r->kernel_sel_sweep = nullptr; r->n_base = 0; r->gen_kernel = nullptr; r->gen_kernel_v1 = nullptr; r->gen_values = 0; r->gen_vec = 0;
  if (precision == 0) { r->kernel = (const void*)k_resident<M_NORMAL1D>; r->n_base = ResValues<M_NORMAL1D>::n_base; }
  if (precision == 0) return pick_block<M_NORMAL1D, double>(block, k);
  if (precision == 1) { set_resident_gen<M_NORMAL1D, float>(r); return pick_block<M_NORMAL1D, float>(block, k); }
  return false;
}

}  // namespace hm
