// inst_binormal2d.cu -- every kernel of model M_BINORMAL2D (its own translation unit: the models build in parallel).
// exp / log coefficients from the constant bank in this translation unit (fastmath.cuh: measured faster for this model)
#define HM_CONST_BANK_COEFFS 1
#include "kernel_sets_impl.cuh"

namespace hm {

bool kernels_binormal2d(int precision, int block, KernelSet* k, ResidentSet* r) {
  r->kernel = nullptr; r->n_base = 0; r->gen_kernel = nullptr; r->gen_values = 0; r->gen_vec = 0;
  if (precision == 0) { set_resident_gen<M_BINORMAL2D, double>(r); return pick_block<M_BINORMAL2D, double>(block, k); }
  return false;
}

}  // namespace hm
