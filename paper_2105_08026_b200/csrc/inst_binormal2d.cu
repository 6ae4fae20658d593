// inst_binormal2d.cu -- every kernel of model M_BINORMAL2D (its own translation unit: the models build in parallel).
// exp / log coefficients from the constant bank in this translation unit (fastmath.cuh: measured faster for this model)
#define HM_CONST_BANK_COEFFS 1
#include "kernel_sets_impl.cuh"

namespace hm {

bool kernels_binormal2d(int precision, int block, KernelSet* k, ResidentSet* r) {
  r->kernel = nullptr; r->kernel_sel_sweep = nullptr; r->n_base = 0; r->gen_kernel = nullptr; r->gen_kernel_v1 = nullptr; r->gen_values = 0; r->gen_vec = 0;
  if (precision == 0) {
    set_resident_gen<M_BINORMAL2D, double>(r);
    if (!pick_block<M_BINORMAL2D, double>(block, k)) return false;
    if (block == 512) {     // p = 2 in fp64: 12 sweep warps with 170 registers are as fast as 16 with 128, which leaves room for tail warps
      k->persistent_dt = (const void*)k_persistent_dt<M_BINORMAL2D, double, 384>;
      k->persistent_dt_nomom = (const void*)k_persistent_dt<M_BINORMAL2D, double, 384, true>;
      k->dt_sweep_threads = 384;
      k->sweep_dt = (const void*)k_sweep<M_BINORMAL2D, double, 384, false>;
      k->sweep_tap_dt = (const void*)k_sweep<M_BINORMAL2D, double, 384, true>;
    }
    return true;
  }
  return false;
}

}  // namespace hm
