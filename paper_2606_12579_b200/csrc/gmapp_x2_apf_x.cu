// gmapp_x2_apf_x.cu -- instantiates the packed f32x2 rollout kernels for 3D point agents: APF (Eq. 1) heuristic, static spheres, with the snapshot / trajectory extras (own translation unit: parallel
// compilation only).
#include "gmapp_tables.h"

namespace gmapp {
rollout_x2_fn rollout_x2_kernel_apf_x(int at, int mode, bool cull, int stage) {
#define PICKX(A, M, MT)                                                                                                                                   \
    (cull ? (stage ? (rollout_x2_fn)k_rollout_x2<A, M, true, 1, MT, true, true, false> : (rollout_x2_fn)k_rollout_x2<A, M, true, 0, MT, true, true, false>)     \
          : (stage ? (rollout_x2_fn)k_rollout_x2<A, M, false, 1, MT, true, true, false> : (rollout_x2_fn)k_rollout_x2<A, M, false, 0, MT, true, true, false>))
    // mode 3 = mode 2 compiled for up to 7 groups (21 warps, 80 registers); mode 2 proper holds <= 4 groups
    // (20 warps = 5 per SM sub-partition, 96 registers), which is what one wave of config 3 needs
    if (mode == 4) return PICKX(2, 4, 512);
    if (at == 2) return mode == 3 ? PICKX(2, 2, 672) : (mode == 2 ? PICKX(2, 2, 640) : (mode == 1 ? PICKX(2, 1, 512) : PICKX(2, 0, 512)));
    return mode == 3 ? PICKX(1, 2, 672) : (mode == 2 ? PICKX(1, 2, 640) : (mode == 1 ? PICKX(1, 1, 512) : PICKX(1, 0, 512)));
#undef PICKX
}
}  // namespace gmapp
