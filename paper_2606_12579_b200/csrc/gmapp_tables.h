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
// One table per translation unit: (agents per group, mode, cull, stage) -> kernel.  stage 2 (TMA tile ring) exists in the
// branch-free form only (cull is an explicit tuning knob; with it, sets beyond shared memory are read through L2).
// mode 2 proper holds <= 4 groups (20 warps = 5 per SM sub-partition, 96 registers), which is what one wave of config 3 needs.
// mode 3 = 5 to 7 groups: with two agents per group (tag MAXT 576) mixed group widths, 16 sweep warps and one epilogue warp per two
// groups (19 or 20 warps, 96 registers);
// with one agent per group (a tuning-only shape) the mode-2 code compiled for 21 warps (80 registers).
#define GMAPP_X2_PICK(A, M, MT, F, X, V)                                                                                     \
    (stage == 2 ? (rollout_x2_fn)k_rollout_x2<A, M, false, 2, MT, F, X, V>                                                  \
     : cull ? (stage ? (rollout_x2_fn)k_rollout_x2<A, M, true, 1, MT, F, X, V> : (rollout_x2_fn)k_rollout_x2<A, M, true, 0, MT, F, X, V>)   \
            : (stage ? (rollout_x2_fn)k_rollout_x2<A, M, false, 1, MT, F, X, V> : (rollout_x2_fn)k_rollout_x2<A, M, false, 0, MT, F, X, V>))
#define GMAPP_X2_PICK01(A, M, MT, F, X, V)                                                                                   \
    (cull ? (stage ? (rollout_x2_fn)k_rollout_x2<A, M, true, 1, MT, F, X, V> : (rollout_x2_fn)k_rollout_x2<A, M, true, 0, MT, F, X, V>)     \
          : (stage ? (rollout_x2_fn)k_rollout_x2<A, M, false, 1, MT, F, X, V> : (rollout_x2_fn)k_rollout_x2<A, M, false, 0, MT, F, X, V>))
#define GMAPP_X2_TABLE(NAME, F, X, V)                                                                                        \
    rollout_x2_fn NAME(int at, int mode, bool cull, int stage) {                                                             \
        if (stage == 2 && (cull || mode == 0)) return nullptr;                                                               \
        if (mode == 4) return GMAPP_X2_PICK(2, 4, 512, F, X, V);                                                             \
        if (mode == 0) {                                                                                                      \
                         return at == 2 ? GMAPP_X2_PICK01(2, 0, 512, F, X, V) : GMAPP_X2_PICK01(1, 0, 512, F, X, V); }       \
        if (at == 2) return mode == 3 ? GMAPP_X2_PICK(2, 2, 576, F, X, V) : (mode == 2 ? GMAPP_X2_PICK(2, 2, 640, F, X, V) : GMAPP_X2_PICK(2, 1, 512, F, X, V)); \
        return mode == 3 ? GMAPP_X2_PICK(1, 2, 672, F, X, V) : (mode == 2 ? GMAPP_X2_PICK(1, 2, 640, F, X, V) : GMAPP_X2_PICK(1, 1, 512, F, X, V));              \
    }
// gmapp_wide.cu: multi-warp groups with epilogue warps for 6D motor agents
rollout_fn rollout_wide_kernel_tu(bool moving, bool cull, int stage, bool apf);
}  // namespace gmapp
