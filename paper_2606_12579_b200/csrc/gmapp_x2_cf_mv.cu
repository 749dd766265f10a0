// gmapp_x2_cf_mv.cu -- instantiates the packed f32x2 rollout kernels for 3D point agents: circular-field (Eq. 2-3) heuristic, moving spheres
// (own translation unit: parallel compilation only; the table macro lives in gmapp_tables.h).
#include "gmapp_tables.h"

namespace gmapp {
GMAPP_X2_TABLE(rollout_x2_kernel_cf_mv, false, false, true)
}  // namespace gmapp
