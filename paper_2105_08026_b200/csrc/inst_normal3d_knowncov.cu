// inst_normal3d_knowncov.cu -- every kernel of model M_NORMAL3D_KNOWNCOV (its own translation unit: the models build in parallel).
#include "kernel_sets_impl.cuh"

namespace hm {

bool kernels_normal3d_knowncov(int precision, int block, KernelSet* k, ResidentSet* r) {
  r->kernel = nullptr; r->kernel_sel_sweep = nullptr; r->n_base = 0; r->gen_kernel = nullptr; r->gen_kernel_v1 = nullptr; r->gen_values = 0; r->gen_vec = 0;
  if (precision == 0) { set_resident_gen<M_NORMAL3D_KNOWNCOV, double>(r); return pick_block<M_NORMAL3D_KNOWNCOV, double>(block, k); }
  return false;
}

}  // namespace hm
