// inst_thinned_schechter1d_selsweep.cu -- k_resident<M_THINNED_SCHECHTER1D, SEL_SWEEP> alone, in a translation unit of its
// own so that it can take its exp / log coefficients from the constant bank (fastmath.cuh: which source is faster depends on
// the kernel).  Same-box A/B on C1: 4.339 -> 4.259 us per iteration; the default instantiation (C2) loses 0.3 % with the same
// switch and stays in inst_thinned_schechter1d.cu with literal coefficients.
#define HM_CONST_BANK_COEFFS 1
// two Newton steps in log / sqrt (fastmath.cuh, HM_NEWTON_STEPS): measured faster for the on-chip p = 1 kernel of this model
#define HM_NEWTON_STEPS 2
#include "kernel_sets_impl.cuh"

namespace hm {

const void* kernel_sel_sweep_thinned_schechter1d() { return (const void*)k_resident<M_THINNED_SCHECHTER1D, true>; }

}  // namespace hm
