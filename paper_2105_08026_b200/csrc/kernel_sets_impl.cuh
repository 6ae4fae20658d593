// kernel_sets_impl.cuh -- included by the per-model translation units inst_*.cu only: instantiates every kernel of
// one model and fills its KernelSet / ResidentSet.
#pragma once
#include "kernel_sets.h"
#include "kernels.cuh"
#include "resident.cuh"
#include "resident_gen.cuh"
#include "stream_tma.cuh"

namespace hm {

template <int MODEL, class T, int BLOCK, bool WITH_TMA = true>
KernelSet make_set() {
  KernelSet k;
  k.persistent = (const void*)k_persistent<MODEL, T, BLOCK, PK_PLAIN>;
  k.persistent_ahead = (const void*)k_persistent<MODEL, T, BLOCK, PK_AHEAD>;
  k.persistent_hold = (const void*)k_persistent<MODEL, T, BLOCK, PK_HOLD>;
  k.sweep_hold = (const void*)k_sweep<MODEL, T, BLOCK, false, true>;
  k.sweep_tap_hold = (const void*)k_sweep<MODEL, T, BLOCK, true, true>;
  k.persistent_dt = nullptr; k.persistent_dt_nomom = nullptr; k.dt_sweep_threads = 0; k.sweep_dt = nullptr; k.sweep_tap_dt = nullptr;
  k.stage_step_bytes = (size_t)DrawSet<MODEL, T>::NV * BLOCK * sizeof(T);
  k.persistent_tma = nullptr;
  if constexpr (WITH_TMA) k.persistent_tma = (const void*)k_persistent_tma<MODEL, T, BLOCK>;
  k.tma_stage_bytes = (size_t)(ModelDims<MODEL>::p * (ModelDims<MODEL>::p + 3) / 2 + ModelDims<MODEL>::ncols) * (BLOCK - 32) * 16;
  k.sweep = (const void*)k_sweep<MODEL, T, BLOCK, false>;
  k.sweep_tap = (const void*)k_sweep<MODEL, T, BLOCK, true>;
  k.init_state = (const void*)k_init_state<MODEL, T>;
  return k;
}

template <int MODEL, class T>
void set_resident_gen(ResidentSet* r) {
  r->gen_kernel = (const void*)k_resident_gen<MODEL, T>;
  r->gen_values = ResGenValues<MODEL, T>::n_values;
  r->gen_vec = VecOf<T>::n;
  r->gen_kernel_v1 = nullptr;
  if constexpr (sizeof(T) == 8 && ModelDims<MODEL>::p >= 2) {
    static_assert(ResGenValues<MODEL, T, 1>::n_values == ResGenValues<MODEL, T>::n_values, "same shared-memory values per object");
    r->gen_kernel_v1 = (const void*)k_resident_gen<MODEL, T, 1>;
  }
}

template <int MODEL, class T>
bool pick_block(int block, KernelSet* k) {
  switch (block) {
    case 256:  *k = make_set<MODEL, T, 256>(); return true;
    case 512:  *k = make_set<MODEL, T, 512>(); return true;
    case 1024: *k = make_set<MODEL, T, 1024>(); return true;
  }
  return false;
}

}  // namespace hm
