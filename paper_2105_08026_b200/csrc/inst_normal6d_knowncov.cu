// inst_normal6d_knowncov.cu -- every kernel of model M_NORMAL6D_KNOWNCOV (its own translation unit: the models build in parallel).
// p = 6: a thread holds two objects of p (p + 5) / 2 doubles each, so only the 256-thread block (255 registers) is built,
// and the TMA-staged variant (one stage of its ring would not fit twice in shared memory) is not.
#include "kernel_sets_impl.cuh"

namespace hm {

bool kernels_normal6d_knowncov(int precision, int block, KernelSet* k, ResidentSet* r) {
  r->kernel = nullptr; r->kernel_sel_sweep = nullptr; r->n_base = 0; r->gen_kernel = nullptr; r->gen_kernel_v1 = nullptr; r->gen_values = 0; r->gen_vec = 0;
  if (precision != 0 || block != 256) return false;
  set_resident_gen<M_NORMAL6D_KNOWNCOV, double>(r);
  *k = make_set<M_NORMAL6D_KNOWNCOV, double, 256, false>();
  return true;
}

}  // namespace hm
