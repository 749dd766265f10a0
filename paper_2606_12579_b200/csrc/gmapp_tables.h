// gmapp_tables.h -- kernel-table functions of the separately compiled translation units (the rollout kernels are
// split over several .cu files only so that nvcc can compile them in parallel; no device code crosses a TU).
#pragma once
#include "gmapp_kernels.cuh"
#include "gmapp_rollout_x2.cuh"

namespace gmapp {
typedef void (*rollout_fn)(const RolloutParams);
typedef void (*rollout_x2_fn)(const RolloutX2Params);
// gmapp_x2_cf.cu / gmapp_x2_apf.cu: packed f32x2 kernels for static spheres, circular field / APF
rollout_x2_fn rollout_x2_kernel_cf(int at, int mode, bool cull, int stage);
rollout_x2_fn rollout_x2_kernel_apf(int at, int mode, bool cull, int stage);
// gmapp_x2_cf_x.cu / gmapp_x2_apf_x.cu: the same with the snapshot / trajectory extras compiled in
rollout_x2_fn rollout_x2_kernel_cf_x(int at, int mode, bool cull, int stage);
rollout_x2_fn rollout_x2_kernel_apf_x(int at, int mode, bool cull, int stage);
// gmapp_wide.cu: multi-warp groups with an epilogue warp for 6D agents and moving spheres
rollout_fn rollout_wide_kernel_tu(int kind, int at, bool moving, bool cull, int stage, bool apf);
}  // namespace gmapp
