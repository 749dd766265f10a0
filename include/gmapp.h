/*
 * gmapp.h -- C ABI of libgmapp.so: the B200 (sm_100a) multi-agent vector-field planner rollout of
 * G-MAPP (arxiv/paper_2606_12579).  "PAPER.md:<n>" cites line n of the paper's text.
 *
 * What the library computes (Sec. IV-A/IV-C, Fig. 2): N_a exploration agents, each a
 * task-space state, are rolled forward N_k steps.  At every step every agent evaluates every obstacle
 * sphere of the sphere world S_W (Eq. 5) with the circular-field / MFI force of Eq. 2-3
 * as gated and clamped by Alg. 1 lines 6-7; the contributions are
 * summed (Alg. 1 lines 10-16), the attractor of Eq. 7-8 is added (Eq. 6), the state
 * is integrated with Eq. 9-11, the costs of Eq. 16-20 are
 * accumulated on the fly, and the best agent is selected.  All of it runs in CUDA
 * kernels; there is no CPU fallback.  Arithmetic is FP32.
 *
 * Conventions
 *  - Every call returns a gmapp_status; nothing throws, aborts or prints.  Arguments, call order and the launch shape
 *    are checked BEFORE the first stream operation: on EINVAL / ECAPACITY / ESTATE nothing has been enqueued, and
 *    gmapp_last_error(ctx) holds a message.  (ECUDA reports a failing CUDA runtime call, wherever it occurs.)
 *  - Coordinates: the sphere world and the agents must stay within 1e5 m of the origin (padding slots of the sphere
 *    arrays are sentinel spheres at (1e6, 1e6, 1e6) with radius 0).
 *  - Pointers named d_* are DEVICE pointers, caller-owned (e.g. torch tensors' data_ptr()), 16-byte
 *    alignment is NOT required.  Pointers named h_* and all struct / scalar-array arguments (goal,
 *    gains, tuning) are HOST pointers, read before the call returns.
 *  - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All calls
 *    are asynchronous on that stream except gmapp_best_agent[_ex], gmapp_select, gmapp_plan_cycle_host,
 *    gmapp_measure_fp32_peak and gmapp_destroy, which synchronise it.  The calls of one planning cycle (rollout,
 *    selection, results) belong on ONE stream; the *_host entry points may be used from different streams (the pinned
 *    staging buffer is guarded by an event).
 *  - The context owns only its packed sphere copy, per-agent result scratch and small pinned staging
 *    buffers, all allocated in gmapp_create (no allocation on the hot path).  One context is not
 *    thread-safe; separate contexts are independent.
 *  - State layouts.  GMAPP_POINT3: [n][6] = (p_x,p_y,p_z, v_x,v_y,v_z), world frame.
 *    GMAPP_MOTOR6: [n][14] = motor[8] + twist[6].  motor = (r_w,r_x,r_y,r_z, d_w,d_x,d_y,d_z), the unit
 *    dual quaternion r + eps d with d = (1/2) t (x) r, t = world translation as a pure quaternion,
 *    r = rotation (Hamilton convention, x_world = R(r) x_body + t): component for component the scalar,
 *    3 rotation-bivector, 3 translation-bivector and pseudoscalar coefficients of a geometric-algebra
 *    motor of Spin(3) |x R^3.  twist = (w_x,w_y,w_z, v_x,v_y,v_z) in the BODY frame
 *    (Eq. 11 right-multiplies).  Input motors are renormalised (|r| = 1, r.d = 0).
 *  - goal: POINT3 3 floats (p_g); MOTOR6 8 floats (goal motor).
 */
#ifndef GMAPP_H
#define GMAPP_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gmapp_ctx gmapp_ctx;   /* opaque */

typedef enum {
    GMAPP_OK = 0,
    GMAPP_EINVAL = 1,      /* NULL pointer, non-positive size, non-finite dt, bad gains (eps<=0, r_d<=0, eps>r_d) */
    GMAPP_ECAPACITY = 2,   /* n exceeds max_agents / max_spheres given to gmapp_create */
    GMAPP_ESTATE = 3,      /* call order: rollout/forces before set_obstacles, best_agent before rollout */
    GMAPP_ECUDA = 4        /* a CUDA runtime call failed; message in gmapp_last_error */
} gmapp_status;

typedef enum {
    GMAPP_POINT3 = 0,      /* 3D point agents: p[3], v[3] */
    GMAPP_MOTOR6 = 1       /* 6D pose agents: motor[8], twist[6] */
} gmapp_kind;

/* Gains and constants (POD, host memory).  Field-by-field meaning and the paper passage:          */
typedef struct {
    float k_circ;          /* k_f of Eq. 2 / Eq. 1; applied once                   */
    float k_att, k_damp;   /* linear (translational) blocks of K and D in Eq. 7       */
    float k_att_rot, k_damp_rot;   /* rotational blocks of K and D, MOTOR6 only                      */
    float inv_mass, inv_inertia;   /* diagonal of the "tunable inertia tensor" of Eq. 9 */
    float vel_factor;      /* the printed 1/2 of Eq. 10; default 0.5                  */
    float r_influence;     /* r_d, detection radius (Eq. 1, Alg. 1 line 7)                           */
    float r_agent;         /* r_a of Alg. 1; default 0                                */
    float eps_dist;        /* epsilon of Alg. 1 line 6; default 1e-3 m                */
    float w_goal, w_obs, w_path, w_smooth;   /* w_j of Eq. 16                         */
    float r_cost_goal, r_cost_obs;           /* radii of Eq. 17 / Eq. 18; 0 => r_influence           */
    float a_max;           /* Eq. 20; default 10 m/s^2                                */
    int32_t heuristic;     /* 0 = circular field / MFI (Eq. 2-3); 1 = APF (Eq. 1)    */
} gmapp_gains;

/* Launch tuning (all 0 / -1 = choose automatically from N_a, N_O and the SM count).               */
typedef struct {
    int32_t lanes_per_agent;     /* threads that share one agent's sphere sum; power of two 1..1024 (packed kernels:
                                    <= 512; with more than 32 agents per CTA only 32 is accepted there)  */
    int32_t agents_per_thread;   /* 1 or 2: agents evaluated per staged sphere load                  */
    int32_t cull;                /* -1 auto, 0 = branch-free force math for every pair,
                                    1 = warp-vote skip of the force math when no lane's pair is inside r_d
                                    (Alg. 1 line 7 is such a branch); results are identical */
    int32_t stage;               /* -1 auto (1 when the set fits; else 2 where the tile ring measures faster than L2 reads:
                                    >= 8 tiles and whole-warp groups; else 0), 0 = read spheres from global memory / L2,
                                    1 = stage the whole sphere set in shared memory by TMA bulk copies (EINVAL when it does
                                    not fit), 2 = stream tiles through a shared-memory ring by TMA bulk copies (packed kernels,
                                    branch-free, groups of >= 32 lanes; EINVAL otherwise)                                   */
    int32_t max_ctas;            /* 0 = SM count; cap on the grid (for scaling experiments)           */
    int32_t scalar_path;         /* 0 = packed f32x2 kernels where they apply (POINT3 in every shape, static and
                                    moving spheres; MOTOR6 agents when a group spans >= 64 lanes and there
                                    are <= 4 groups per CTA); 1 = force the scalar FP32 kernel (A/B)    */
    int32_t reserved[2];
} gmapp_tuning;

/* What the last gmapp_rollout launched (for reporting). */
typedef struct {
    int32_t grid, block;
    int32_t lanes_per_agent, agents_per_thread, agents_per_cta;
    int32_t cull, stage, tile_spheres, n_tiles;
    int32_t smem_bytes, regs_per_thread;
    int32_t kernels_launched;    /* kernels this call enqueued */
    int32_t packed_x2;           /* 1 = the packed f32x2 kernel ran, 0 = the scalar kernel */
    int32_t selection_fused;     /* 1 = the selection ran in the tail of the rollout kernel (wide 6D kernel), 0 = gmapp_best_agent
                                    launches the selection kernel behind the rollout (programmatic stream serialisation) */
} gmapp_launch_info;

/* Fill *g with the defaults listed above (k_circ 1, k_att 2, k_damp 0.5, rot 2 / 0.5, inv 1, 1/2,
 * r_d 0.15, r_a 0, eps 1e-3, weights 1, cost radii 0, a_max 10, heuristic 0). */
void gmapp_default_gains(gmapp_gains* g);

/* Create a context on CUDA device `device` able to hold max_agents agents and max_spheres spheres.
 * Allocates all device / pinned memory the library will ever use for this context. */
gmapp_status gmapp_create(gmapp_ctx** out, int device, int max_agents, int max_spheres);

/* Synchronises the device work of this context and frees it.  NULL is OK. */
gmapp_status gmapp_destroy(gmapp_ctx* ctx);

/* Load the sphere world S_W (Eq. 5; resident on the GPU).
 * d_xyzr [n][4] = centre xyz + radius (per-sphere radii, a superset of the paper's single r_O);
 * d_vel [n][3] = constant sphere velocities or NULL for a static world.  n = 0 is legal (no obstacles).
 * The arrays are read by stream work enqueued in this call (a packing kernel); they may be freed or
 * changed once that work has run.  Radii must be >= 0 and all values finite (not checked on device). */
gmapp_status gmapp_set_obstacles(gmapp_ctx* ctx, const float* d_xyzr, const float* d_vel, int n, void* cuda_stream);
/* Same with HOST arrays: copied into the context's pinned buffer, which the packing kernel then reads over the host
 * link itself (no device staging copy).  Waits first (on an event, whatever stream it was) for the packing kernel of an
 * earlier host call that may still be reading that buffer. */
gmapp_status gmapp_set_obstacles_host(gmapp_ctx* ctx, const float* h_xyzr, const float* h_vel, int n, void* cuda_stream);

/* Sphere-world builder (perception stage: workspace crop, "voxelise at 2 r_O", the occupied
 * voxel centres are the spheres of S_W, Eq. 5; S_W stays in GPU memory).  d_points [n][3]
 * DEVICE point cloud (world frame; NaN / out-of-box points are dropped); lo, hi: HOST float[3] workspace box
 * (lo <= p < hi); pitch = 2 r_O.  Voxel index floor((p - lo) / pitch) in FP32; the spheres are the occupied voxels in
 * increasing linear voxel index (z-major, then y, then x) with centre lo + (i + 1/2) pitch and radius pitch / 2.
 * The context's sphere world becomes `capacity` static slots: the first min(count, capacity) are those spheres, the
 * rest far-away sentinels that never act -- so no count has to come back to the host; d_count_out (nullable DEVICE
 * int32) receives the number of occupied voxels (> capacity means the tail was dropped).  The packed rollout kernels
 * read that count on the device and sweep only the real spheres.  Asynchronous.  Errors:
 * EINVAL for bad arguments, ECAPACITY for capacity > max_spheres, > 4096 voxels per axis or > 2^25 voxels. */
gmapp_status gmapp_build_sphere_world(gmapp_ctx* ctx, const float* d_points, int n_points, const float* lo,
                                      const float* hi, float pitch, int capacity, int32_t* d_count_out,
                                      void* cuda_stream);

/* ALLOCATION-FREE variant of the sphere-world builder, for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it).  No context: the scratch memory (voxel bitmap + block
 * counter) is a file-scope static device array of the library -- 33 024 bytes that every GPU that loads the library
 * holds until the process exits -- and the call performs no cudaMalloc / cudaFree / allocating library routine.
 * Same computation and conventions as gmapp_build_sphere_world (Eq. 5); the result
 * goes to the CALLER's DEVICE buffer d_xyzr_out [capacity][4] (16-byte aligned): the min(count, capacity) occupied-voxel
 * spheres (x, y, z, r) in increasing linear voxel index, then sentinels (1e6, 1e6, 1e6, 0) -- i.e. what
 * gmapp_build_sphere_world + gmapp_get_obstacles return, bit for bit; d_count_out (nullable DEVICE int32) = occupied voxels.
 * Feed it to gmapp_set_obstacles.  LIMIT: the voxel grid may hold at most 262 144 voxels (e.g. 64^3; the paper's 1 m^3
 * workspace at pitch 4 cm has 15 625) and 4096 per axis; larger grids return GMAPP_ECAPACITY with nothing launched
 * (use gmapp_build_sphere_world).  `device` = CUDA device index 0..63, made current by the call.  Asynchronous on
 * cuda_stream (a memset of the scratch, then one kernel).  All calls on a device SHARE the one scratch array (it is cleared
 * at the start of every call): calls whose stream work overlaps on the same GPU race -- keep them on one stream or order them.
 * Errors: EINVAL / ECAPACITY / ECUDA; the message is in gmapp_last_error(NULL). */
gmapp_status gmapp_build_sphere_world_static(int device, const float* d_points, int n_points, const float* lo,
                                             const float* hi, float pitch, int capacity, float* d_xyzr_out,
                                             int32_t* d_count_out, void* cuda_stream);

/* Copy the first n spheres of the resident sphere world, (x, y, z, r) each, into a caller-owned DEVICE buffer
 * [n][4] (after gmapp_build_sphere_world: the occupied-voxel spheres, then sentinels at (1e6, 1e6, 1e6) with radius 0).  Asynchronous. */
gmapp_status gmapp_get_obstacles(gmapp_ctx* ctx, float* d_xyzr_out, int n, void* cuda_stream);

/* Optional launch tuning for later gmapp_rollout calls (gmapp_forces has one launch shape and ignores it); NULL restores
 * the automatic choice. */
gmapp_status gmapp_set_tuning(gmapp_ctx* ctx, const gmapp_tuning* tuning);

/* Heterogeneous ensemble ("two agents per heuristic type, each with either a large or small
 * detection radius"; Alg. 1 takes r_d per agent; one specialised kernel per heuristic,
 * PAPER.md:262-266).  HOST arrays of n values, any of them NULL (= take the value from `gains`):
 * h_r_influence[i] = r_d of agent i (> 0), h_k_circ[i] = k_f of agent i, h_heuristic[i] in {0 = circular field /
 * MFI (Eq. 2-3), 1 = APF (Eq. 1)}.  The arrays are copied into the context's pinned staging buffer before the call returns and go
 * to the device by asynchronous copies on cuda_stream (an earlier call's copies, on whatever stream, are waited for first).
 * Later gmapp_rollout calls must pass n_agents == n (else EINVAL); they issue one launch per heuristic present,
 * and the Eq. 17 / 18 radii default to each agent's own r_d.  n = 0 (or all three NULL) restores uniform agents.
 * gmapp_forces keeps using `gains` alone (it ignores these arrays). */
gmapp_status gmapp_set_agent_params(gmapp_ctx* ctx, const float* h_r_influence, const float* h_k_circ,
                                    const int32_t* h_heuristic, int n, void* cuda_stream);

/* One planning cycle: roll n_agents agents forward `steps` steps of size dt from the
 * states in d_agents (layout by `kind`), through Eq. 2-3, 6-11, accumulating Eq. 16-20 over the
 * steps+1 poses.  Final states are written to d_agents_out (same layout; may alias d_agents; may be
 * NULL).  Per-agent costs / clearance / collision flags stay in the context (gmapp_get_results,
 * gmapp_best_agent).  Obstacles move as c_j(t) = c_j + t u_j, t = k dt at step k.
 * Errors: EINVAL for NULL / n_agents < 1 / steps < 1 / non-finite or non-positive dt / bad gains;
 * ECAPACITY for n_agents > max_agents; ESTATE before gmapp_set_obstacles. */
gmapp_status gmapp_rollout(gmapp_ctx* ctx, gmapp_kind kind, const float* d_agents, float* d_agents_out,
                           int n_agents, const float* goal, const gmapp_gains* gains, float dt, int steps,
                           void* cuda_stream);

/* Explored paths (PAPER.md:51 lists them among the planner's outputs; Eq. 15): while d_traj is set,
 * every gmapp_rollout also writes all steps+1 poses of every agent to the caller-owned DEVICE buffer
 * d_traj [n_agents][steps+1][6|14] (same state layout as the agents; pose 0 is the start state as given).  The buffer
 * must hold the largest later rollout.  NULL switches it off (the default).  One 24- or 56-byte store per agent-step. */
gmapp_status gmapp_set_trajectory_output(gmapp_ctx* ctx, float* d_traj);

/* Closed-loop re-planning (Fig. 2 steps 3-5: the planner re-plans from the robot's state while
 * the control thread follows the best agent).  n_cycles planning cycles are chained ON THE DEVICE, nothing
 * synchronises: cycle c rolls all agents `steps` steps from d_agents (obstacles at time c * exec_steps * dt),
 * selects the best agent with hysteresis against the previous cycle's winner (prev_best for the first cycle, < 0 =
 * none), takes that agent's state after exec_steps steps as the robot's new state -- following the winning
 * agent's own control law for exec_steps steps IS that agent's rollout truncated there -- and restarts every agent
 * from it (ensemble diversity then comes from gmapp_set_agent_params).  d_agents [n][6|14] is read and overwritten
 * (after the call it holds the last robot state, replicated); d_path_out [n_cycles][6|14] (nullable) receives the
 * robot state after each cycle, d_best_out [n_cycles] int32 (nullable) the winners.  Asynchronous on the stream;
 * capturable in a CUDA graph.  Errors: EINVAL for NULL / n_cycles < 1 / exec_steps outside 1..steps, plus every
 * error of gmapp_rollout. */
gmapp_status gmapp_replan(gmapp_ctx* ctx, gmapp_kind kind, float* d_agents, int n_agents, const float* goal,
                          const gmapp_gains* gains, float dt, int steps, int exec_steps, float alpha, int prev_best,
                          int n_cycles, float* d_path_out, int32_t* d_best_out, void* cuda_stream);

/* Agent selection: lexicographic argmin of (collided, C_i, i) over the last rollout;
 * with prev_best >= 0 the incumbent keeps its place unless the challenger is collision-free while the
 * incumbent collided, or the flags are equal and C_best < alpha * C_prev.  A NaN cost ranks last.
 * Synchronises the stream and returns index and cost to host memory.
 * The reduction itself runs in the TAIL of the rollout kernel (the warp that finishes the last agent reduces all
 * agents' keys and writes the record to pinned host memory): with prev_best < 0, or with the (alpha, prev_best) the
 * rollout was armed with by gmapp_set_selection, this call only synchronises and reads that record -- no second launch
 * in the planning cycle.  With other arguments (and after the scalar kernels, which have no such tail) a small
 * selection kernel is launched.  prev_best >= n_agents of the last rollout counts as "no incumbent".  Errors: ESTATE
 * before any rollout, EINVAL for non-finite alpha. */
gmapp_status gmapp_best_agent(gmapp_ctx* ctx, float alpha, int prev_best, int* out_index, float* out_cost,
                              void* cuda_stream);

/* Same, and also returns the winner's collision flag (needed to merge winners of several GPUs, each
 * of which rolled its own block of agents). */
gmapp_status gmapp_best_agent_ex(gmapp_ctx* ctx, float alpha, int prev_best, int* out_index, float* out_cost,
                                 int* out_collided, void* cuda_stream);

/* The full selection record of the last rollout for (alpha, prev_best): the selected agent, the plain argmin without
 * incumbent, and the incumbent's own key this cycle (what several GPUs exchange to apply the hysteresis rule once,
 * globally).  Same cost and synchronisation as gmapp_best_agent. */
typedef struct {
    int32_t index, collided; float cost;              /* selected agent (hysteresis applied)                      */
    int32_t raw_index, raw_collided; float raw_cost;  /* lexicographic argmin of (collided, C, index), no incumbent */
    int32_t prev_collided; float prev_cost;           /* the incumbent's key (valid when prev_best >= 0)          */
} gmapp_selection;
gmapp_status gmapp_select(gmapp_ctx* ctx, float alpha, int prev_best, gmapp_selection* out, void* cuda_stream);

/* Arm the selection that later gmapp_rollout calls fuse into their tail: hysteresis factor alpha and incumbent prev_best
 * (< 0 = none, the default; an index beyond a later rollout's agents counts as none).  gmapp_plan_cycle_host and
 * gmapp_replan arm it themselves.  EINVAL for non-finite alpha or prev_best >= max_agents. */
gmapp_status gmapp_set_selection(gmapp_ctx* ctx, float alpha, int prev_best);

/* Force query without integration (the control thread's query, Fig. 2 step 5):
 * for each state, d_f_rep [n][3] = sum_j f_j (world frame, Eq. 2-3 / Alg. 1) with obstacles at time
 * t_obstacles, and d_f_total = Eq. 6: POINT3 [n][3] = f_a + f_r; MOTOR6 [n][6] = body wrench
 * (torque, force).  Either output may be NULL. */
gmapp_status gmapp_forces(gmapp_ctx* ctx, gmapp_kind kind, const float* d_agents, int n_agents, const float* goal,
                          const gmapp_gains* gains, float t_obstacles, float* d_f_rep, float* d_f_total,
                          void* cuda_stream);

/* Copy the per-agent results of the last rollout into caller-owned DEVICE buffers (any may be NULL):
 * d_cost [n][5] = {C, C_goal, C_obs, C_path, C_smooth} (Eq. 16-20); d_min_clearance [n] = min over poses
 * and spheres of the surface distance (+inf with no obstacles); d_collided [n] int32. */
gmapp_status gmapp_get_results(gmapp_ctx* ctx, float* d_cost, float* d_min_clearance, int32_t* d_collided,
                               void* cuda_stream);

/* A whole planning cycle from HOST buffers: (optional) sphere upload, agent states read by the rollout kernel straight
 * from the pinned buffer (and final states written back to it), selection in the rollout's tail, its record written to
 * pinned memory; h_agents_out (may be NULL) receives the final states.
 * n_spheres < 0 keeps the resident sphere world (ESTATE if there is none); n_spheres == 0 sets an EMPTY world (no
 * obstacles); n_spheres > 0 uploads h_xyzr [n][4] (+ h_vel [n][3] or NULL).  Synchronises the stream. */
gmapp_status gmapp_plan_cycle_host(gmapp_ctx* ctx, gmapp_kind kind, const float* h_agents, float* h_agents_out,
                                   int n_agents, const float* h_xyzr, const float* h_vel, int n_spheres,
                                   const float* goal, const gmapp_gains* gains, float dt, int steps,
                                   float alpha, int prev_best, int* out_index, float* out_cost,
                                   void* cuda_stream);

/* What the last gmapp_rollout launched. */
gmapp_status gmapp_get_launch_info(const gmapp_ctx* ctx, gmapp_launch_info* out);

/* Measure this GPU's FP32 FMA throughput with a register-only FFMA microkernel (8 independent chains
 * per thread, all SMs), timed with CUDA events on `cuda_stream`; *out_tflops = 2 * FMAs / time.
 * use_f32x2 != 0 issues packed fma.rn.f32x2 instead.  Synchronises. */
gmapp_status gmapp_measure_fp32_peak(gmapp_ctx* ctx, int use_f32x2, float* out_tflops, void* cuda_stream);

/* Issue-cost microbenchmarks behind the instruction-mix reasoning of DESIGN.md section 6 (results: profiles/r02_microbench.md):
 * register-only kernels, 4 warps per SM sub-partition, 8 independent chains of ONE instruction kind.  *out_cycles = SM
 * cycles per warp-instruction per sub-partition at the device's maximum SM clock.  kind: 0 FFMA (three distinct
 * registers), 1 FFMA2 three distinct register pairs, 2 FFMA2 two distinct, 3 FFMA2 with a broadcast operand, 4 MUFU.RCP,
 * 5 MUFU.RCP predicated off on every lane, 6 FMNMX, 7 FMNMX3, 8 FSETP + FSEL (per pair), 9 FFMA2 with three distinct register
 * pairs none of which is shared between chains, 10 FFMA2 + FMNMX (per pair), 11 FFMA2 + 2 FMNMX (per triple), 12 FFMA + FMNMX
 * (per pair), 13 the raw sweep's instruction mix (value x 2 = cycles per agent-trip group), 14 the same mix with scalar FFMA.
 * Synchronises.  EINVAL otherwise. */
gmapp_status gmapp_microbench(gmapp_ctx* ctx, int kind, float* out_cycles, void* cuda_stream);

/* Number of SMs of the context's device. */
int gmapp_sm_count(const gmapp_ctx* ctx);

/* Message of the last failing call on this context (context-owned string, never freed by the caller);
 * with ctx == NULL, the message of the last failing gmapp_create. */
const char* gmapp_last_error(const gmapp_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* GMAPP_H */
