// resident_cfg.h -- launch-shape constants the host (cudahm.cu) shares with the kernels of resident.cuh / stream_tma.cuh.
#pragma once

namespace hm {

constexpr int RES_SW = 16;                          // sweep warps per block of the on-chip kernel
constexpr int RES_S = RES_SW * 32;                  // sweep threads per block
constexpr int RES_TW = 4;                           // tail warps per block (tail_block needs exactly 4)
constexpr int RES_THREADS = RES_S + RES_TW * 32;    // 640
// the general on-chip kernel (resident_gen.cuh): fewer sweep warps, more registers per thread (p >= 2 needs them)
constexpr int RG_SW = 8, RG_S = RG_SW * 32, RG_TW = 4, RG_THREADS = RG_S + RG_TW * 32;   // 384
constexpr int RES_MAX_SMEM = 200 * 1024;            // dynamic shared memory the on-chip kernel may ask for
constexpr int TMA_MAX_STAGES = 4;                   // depth of the TMA ring of k_persistent_tma

}  // namespace hm
