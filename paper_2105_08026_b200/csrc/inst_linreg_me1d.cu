// inst_linreg_me1d.cu -- every kernel of model M_LINREG_ME1D (its own translation unit: the models build in parallel).
#include "kernel_sets_impl.cuh"

namespace hm {

bool kernels_linreg_me1d(int precision, int block, KernelSet* k, ResidentSet* r) {
  r->kernel = nullptr; r->kernel_sel_sweep = nullptr; r->n_base = 0; r->gen_kernel = nullptr; r->gen_kernel_v1 = nullptr; r->gen_values = 0; r->gen_vec = 0;
  if (precision == 0) { r->kernel = (const void*)k_resident<M_LINREG_ME1D>; r->n_base = ResValues<M_LINREG_ME1D>::n_base; }
  if (precision == 0) return pick_block<M_LINREG_ME1D, double>(block, k);
  // (dedicated tail warps, k_persistent_dt, measured SLOWER for the fp32 kernel: 63.4 against 60.9 us on C4 -- it is issue-bound
  // and needs all 16 sweep warps)
  if (precision == 1) { set_resident_gen<M_LINREG_ME1D, float>(r); return pick_block<M_LINREG_ME1D, float>(block, k); }
  return false;
}

}  // namespace hm
