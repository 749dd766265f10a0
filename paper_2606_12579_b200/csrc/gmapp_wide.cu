// gmapp_wide.cu -- instantiates the wide rollout kernels (6D agents, moving spheres; own translation unit: parallel
// compilation only).
#include "gmapp_tables.h"
#include "gmapp_rollout_wide.cuh"

namespace gmapp {
rollout_fn rollout_wide_kernel_tu(int kind, int at, bool moving, bool cull, int stage, bool apf) {
#define PICKS(K, A, M, F)                                                                                             \
    (cull ? (stage ? (rollout_fn)k_rollout_wide<K, A, M, true, 1, F> : (rollout_fn)k_rollout_wide<K, A, M, true, 0, F>)    \
          : (stage ? (rollout_fn)k_rollout_wide<K, A, M, false, 1, F> : (rollout_fn)k_rollout_wide<K, A, M, false, 0, F>))
#define PICKW(K, A, M) (apf ? PICKS(K, A, M, true) : PICKS(K, A, M, false))
    if (kind == 1) return moving ? PICKW(1, 1, true) : PICKW(1, 1, false);
    if (at == 2) return PICKW(0, 2, true);
    return PICKW(0, 1, true);
#undef PICKW
#undef PICKS
}
}  // namespace gmapp
