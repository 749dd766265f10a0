// gmapp_x2_apf_x_mv.cu -- instantiates the packed f32x2 rollout kernels for 3D point agents: APF (Eq. 1) heuristic, moving spheres, with the snapshot / trajectory extras
// (own translation unit: parallel compilation only; the table macro lives in gmapp_tables.h).
#include "gmapp_tables.h"

namespace gmapp {
GMAPP_X2_TABLE(rollout_x2_kernel_apf_x_mv, true, true, true)
}  // namespace gmapp
