// gmapp_wide.cu -- instantiates the wide rollout kernels for 6D motor agents (own translation unit: parallel compilation only).
#include "gmapp_tables.h"
#include "gmapp_rollout_wide.cuh"

namespace gmapp {
rollout_fn rollout_wide_kernel_tu(bool moving, bool cull, int stage, bool apf) {
#define PICKS(M, F)                                                                                                   \
    (cull ? (stage ? (rollout_fn)k_rollout_wide<M, true, 1, F> : (rollout_fn)k_rollout_wide<M, true, 0, F>)    \
          : (stage ? (rollout_fn)k_rollout_wide<M, false, 1, F> : (rollout_fn)k_rollout_wide<M, false, 0, F>))
#define PICKW(M) (apf ? PICKS(M, true) : PICKS(M, false))
    return moving ? PICKW(true) : PICKW(false);
#undef PICKW
#undef PICKS
}
}  // namespace gmapp
