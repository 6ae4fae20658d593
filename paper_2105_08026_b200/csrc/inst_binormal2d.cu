// inst_binormal2d.cu -- every kernel of model M_BINORMAL2D (its own translation unit: the models build in parallel).
#include "kernel_sets_impl.cuh"

namespace hm {

bool kernels_binormal2d(int precision, int block, KernelSet* k, ResidentSet* r) {
  r->kernel = nullptr; r->n_base = 0;
  if (precision == 0) return pick_block<M_BINORMAL2D, double>(block, k);
  return false;
}

}  // namespace hm
