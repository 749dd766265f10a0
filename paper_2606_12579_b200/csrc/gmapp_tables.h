// gmapp_tables.h -- kernel-table functions of the separately compiled translation units (the rollout kernels are
// split over several .cu files only so that nvcc can compile them in parallel; no device code crosses a TU).
#pragma once
#include "gmapp_kernels.cuh"
#include "gmapp_rollout_x2.cuh"

namespace gmapp {
typedef void (*rollout_fn)(const RolloutParams);
typedef void (*rollout_x2_fn)(const RolloutX2Params);
// gmapp_x2_<cf|apf>[_x][_mv].cu: packed f32x2 kernels for 3D point agents; circular field / APF, plain / with the
// snapshot and trajectory extras, static / moving spheres
rollout_x2_fn rollout_x2_kernel_cf(int at, int mode, bool cull, int stage);
rollout_x2_fn rollout_x2_kernel_cf_x(int at, int mode, bool cull, int stage);
rollout_x2_fn rollout_x2_kernel_apf(int at, int mode, bool cull, int stage);
rollout_x2_fn rollout_x2_kernel_apf_x(int at, int mode, bool cull, int stage);
rollout_x2_fn rollout_x2_kernel_cf_mv(int at, int mode, bool cull, int stage);
rollout_x2_fn rollout_x2_kernel_cf_x_mv(int at, int mode, bool cull, int stage);
rollout_x2_fn rollout_x2_kernel_apf_mv(int at, int mode, bool cull, int stage);
rollout_x2_fn rollout_x2_kernel_apf_x_mv(int at, int mode, bool cull, int stage);
// gmapp_wide.cu: multi-warp groups with epilogue warps for 6D motor agents
rollout_fn rollout_wide_kernel_tu(bool moving, bool cull, int stage, bool apf);
}  // namespace gmapp
