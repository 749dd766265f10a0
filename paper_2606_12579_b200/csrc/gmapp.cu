// gmapp.cu -- host side of libgmapp.so: context, argument validation, launch selection and the
// extern "C" entry points declared in include/gmapp.h.  No torch types; plain CUDA runtime.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#define GMAPP_MAIN_TU
#include "../../include/gmapp.h"
#include "gmapp_kernels.cuh"
#include "gmapp_rollout_x2.cuh"
#include "gmapp_tables.h"
#include "gmapp_voxel.cuh"
#include "gmapp_microbench.cuh"

using namespace gmapp;

struct gmapp_ctx {
    int device = 0, num_sms = 0, smem_optin = 0;
    int max_agents = 0, max_spheres = 0, cap_spheres = 0;
    // packed sphere world: raw radii, and radii + r_agent (only materialised when r_agent != 0)
    float4* d_sph_raw = nullptr;
    float4* d_sph_eff = nullptr;
    float4* d_svel = nullptr;
    // sphere-pair layout of the packed f32x2 rollout kernel: (cx0,cx1,cy0,cy1), (cz0,cz1,-R0,-R1), R = r + r_agent
    float4* d_pairA = nullptr;
    float4* d_pairB = nullptr;
    float pair_r_agent = 0.0f;
    bool pair_valid = false;
    float* d_sph_stats = nullptr;        // {largest R = r_j + r_agent, largest sphere speed} of the pair arrays (tile ring)
    bool stats_valid = false;
    float eff_r_agent = 0.0f;
    bool eff_valid = false;
    int n_spheres = -1;            // -1: set_obstacles not called yet
    bool moving = false;
    // per-agent results of the last rollout
    float* d_cost = nullptr; float* d_minclr = nullptr; int* d_collided = nullptr;
    int last_n_agents = 0;
    // staging for the *_host entry points
    float* h_pinned = nullptr;           // spheres*7 + agents*14 floats
    size_t h_pinned_floats = 0;
    // heterogeneous ensemble (gmapp_set_agent_params): per-agent r_d, k_f, and agent indices grouped by heuristic
    float* d_ap_rd = nullptr; float* d_ap_kf = nullptr; int* d_ap_idx = nullptr;
    float* h_ap = nullptr;               // pinned staging: 3 * max_agents words
    int ap_n = 0;                        // 0: not set
    bool ap_has_rd = false, ap_has_kf = false, ap_has_h = false;
    int ap_count[2] = {0, 0};            // agents per heuristic; d_ap_idx holds class 0 first, then class 1
    float ap_min_rd = 0.0f;
    const int* sub_idx = nullptr;        // the sub-launch being issued (one per heuristic)
    // sphere-world builder (gmapp_build_sphere_world): voxel bitmap (2^25 voxels), block sums, occupied-voxel count
    unsigned* d_vox_bitmap = nullptr; int* d_vox_count = nullptr;
    unsigned long long* d_vox_state = nullptr; int* d_vox_sync = nullptr;      // scan state of k_vox_compact (zero between builds)
    // closed-loop re-planning (gmapp_replan)
    float* d_snap = nullptr;             // [max_agents][14]
    int* d_prev = nullptr;               // incumbent on the device
    float roll_t0 = 0.0f; float* roll_snap = nullptr; int roll_snap_step = 0;
    float* roll_traj = nullptr;          // trajectory output of the next rollouts (gmapp_set_trajectory_output)
    bool built_world = false;            // the sphere world came from gmapp_build_sphere_world: its count lives in d_vox_count
    // selection (S8): the 8-word record {index, collided, cost | raw index, raw collided, raw cost | incumbent collided,
    // cost} on the device and in pinned host memory, and the ticket counter of the rollout kernels' fused tail
    int* d_sel_rec = nullptr; int* d_sel_ticket = nullptr;
    int* h_best = nullptr;               // pinned: the record
    float sel_alpha = 0.9f; int sel_prev = -1;      // what later rollouts' tails are armed with (gmapp_set_selection)
    const int* sel_prev_dev = nullptr;   // gmapp_replan: the incumbent lives on the device
    bool sel_want = false;               // the rollout being issued may fuse the selection into its launches
    bool sel_fused = false;              // the last rollout did: the record holds (fused_alpha, fused_prev)'s selection
    float fused_alpha = 0.0f; int fused_prev = -1; bool fused_prev_dev = false;
    int sel_total = 0;
    int sel_seq = 0;                     // sequence number of the last rollout's selection record (the host polls pinned memory for it)
    cudaEvent_t ev_pinned = nullptr;     // after the last kernel that reads the pinned sphere staging buffer
    bool pinned_busy = false;
    cudaEvent_t ev_ap = nullptr;         // after the last copy out of the pinned per-agent-parameter staging buffer h_ap
    bool ap_busy = false;
    float* d_scratch = nullptr;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    gmapp_tuning tuning;
    bool has_tuning = false;
    gmapp_launch_info info;
    char err[512];
};

static char g_create_err[512] = "";

static gmapp_status fail(gmapp_ctx* c, gmapp_status s, const char* fmt, const char* a = "", long x = 0, long y = 0) {
    char* dst = c ? c->err : g_create_err;
    snprintf(dst, 512, fmt, a, x, y);
    return s;
}
#define CUDA_TRY(ctx, call)                                                                     \
    do {                                                                                        \
        cudaError_t e__ = (call);                                                               \
        if (e__ != cudaSuccess) return fail(ctx, GMAPP_ECUDA, "CUDA error '%s' at line %ld", cudaGetErrorString(e__), __LINE__); \
    } while (0)

static int round_up(int x, int m) { return (x + m - 1) / m * m; }
static int pow2_floor(int x) { int p = 1; while (2 * p <= x) p *= 2; return p; }
static int pow2_ceil(int x) { int p = 1; while (p < x) p *= 2; return p; }
static int ilog2(int x) { int l = 0; while ((1 << l) < x) ++l; return l; }

extern "C" void gmapp_default_gains(gmapp_gains* g) {
    if (!g) return;
    g->k_circ = 1.0f; g->k_att = 2.0f; g->k_damp = 0.5f; g->k_att_rot = 2.0f; g->k_damp_rot = 0.5f;
    g->inv_mass = 1.0f; g->inv_inertia = 1.0f; g->vel_factor = 0.5f;
    g->r_influence = 0.15f; g->r_agent = 0.0f; g->eps_dist = 1e-3f;
    g->w_goal = g->w_obs = g->w_path = g->w_smooth = 1.0f;
    g->r_cost_goal = 0.0f; g->r_cost_obs = 0.0f; g->a_max = 10.0f; g->heuristic = 0;
}

// ---------------------------------------------------------------------------------------------
// kernel table
// ---------------------------------------------------------------------------------------------
// index: kind(2) x at(2: AT=1,2) x moving(2) x cull(2) x stage(2)
static rollout_fn rollout_kernel(int kind, int at, bool moving, bool cull, int stage) {
#define PICK(K, A, MT)                                                                            \
    (moving ? (cull ? (stage ? (rollout_fn)k_rollout<K, A, true, true, 1, MT> : (rollout_fn)k_rollout<K, A, true, true, 0, MT>)      \
                    : (stage ? (rollout_fn)k_rollout<K, A, true, false, 1, MT> : (rollout_fn)k_rollout<K, A, true, false, 0, MT>))   \
            : (cull ? (stage ? (rollout_fn)k_rollout<K, A, false, true, 1, MT> : (rollout_fn)k_rollout<K, A, false, true, 0, MT>)    \
                    : (stage ? (rollout_fn)k_rollout<K, A, false, false, 1, MT> : (rollout_fn)k_rollout<K, A, false, false, 0, MT>)))
    if (kind == GMAPP_MOTOR6) return PICK(1, 1, 512);
    if (at == 2) return PICK(0, 2, 512);
    return PICK(0, 1, 1024);
#undef PICK
}
static const int kX2SweepThreads = 512;       // sweep threads per CTA; mode 2 adds one epilogue warp per group (<= 672 in all)
static rollout_x2_fn rollout_x2_kernel(int at, int mode, bool cull, int stage, bool apf, bool extras, bool moving) {
    if (moving) {
        if (extras) return apf ? gmapp::rollout_x2_kernel_apf_x_mv(at, mode, cull, stage) : gmapp::rollout_x2_kernel_cf_x_mv(at, mode, cull, stage);
        return apf ? gmapp::rollout_x2_kernel_apf_mv(at, mode, cull, stage) : gmapp::rollout_x2_kernel_cf_mv(at, mode, cull, stage);
    }
    if (extras) return apf ? gmapp::rollout_x2_kernel_apf_x(at, mode, cull, stage) : gmapp::rollout_x2_kernel_cf_x(at, mode, cull, stage);
    return apf ? gmapp::rollout_x2_kernel_apf(at, mode, cull, stage) : gmapp::rollout_x2_kernel_cf(at, mode, cull, stage);
}
static rollout_fn rollout_wide_kernel(bool moving, bool cull, int stage, bool apf) {
    return gmapp::rollout_wide_kernel_tu(moving, cull, stage, apf);
}
static int rollout_max_threads(int kind, int at) { return (kind == GMAPP_MOTOR6 || at == 2) ? 512 : 1024; }

// ---------------------------------------------------------------------------------------------
// create / destroy
// ---------------------------------------------------------------------------------------------
extern "C" gmapp_status gmapp_create(gmapp_ctx** out, int device, int max_agents, int max_spheres) {
    if (!out) return fail(nullptr, GMAPP_EINVAL, "gmapp_create: out is NULL%s");
    *out = nullptr;
    if (max_agents < 1 || max_spheres < 0) return fail(nullptr, GMAPP_EINVAL, "gmapp_create: max_agents must be >= 1 and max_spheres >= 0%s");
    int ndev = 0;
    CUDA_TRY(nullptr, cudaGetDeviceCount(&ndev));
    if (device < 0 || device >= ndev) return fail(nullptr, GMAPP_EINVAL, "gmapp_create: no CUDA device %s%ld", "", device);
    CUDA_TRY(nullptr, cudaSetDevice(device));
    gmapp_ctx* c = new gmapp_ctx();
    memset(&c->tuning, 0, sizeof c->tuning);
    memset(&c->info, 0, sizeof c->info);
    c->err[0] = 0;
    c->device = device; c->max_agents = max_agents; c->max_spheres = max_spheres;
    c->cap_spheres = round_up(max_spheres > 0 ? max_spheres : 1, 2048);
    cudaDeviceProp prop;
    cudaError_t e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess) { delete c; return fail(nullptr, GMAPP_ECUDA, "cudaGetDeviceProperties: %s", cudaGetErrorString(e)); }
    if (prop.major < 10) { delete c; return fail(nullptr, GMAPP_ECUDA, "libgmapp is built for sm_100a only; device is sm_%s%ld%ld", "", prop.major, prop.minor); }
    c->num_sms = prop.multiProcessorCount;
    c->smem_optin = (int)prop.sharedMemPerBlockOptin;
    // pinned staging: [0, 7*cap) spheres (xyzr then vel), [7*cap, 7*cap + 14*max_agents) agents
    size_t hp = (size_t)c->cap_spheres * 7 + (size_t)max_agents * 14;
    c->h_pinned_floats = hp;
#define ALLOC(p, bytes) if ((e = cudaMalloc((void**)&(p), (bytes))) != cudaSuccess) { gmapp_destroy(c); return fail(nullptr, GMAPP_ECUDA, "cudaMalloc: %s", cudaGetErrorString(e)); }
    ALLOC(c->d_sph_raw, sizeof(float4) * c->cap_spheres);
    ALLOC(c->d_sph_eff, sizeof(float4) * c->cap_spheres);
    ALLOC(c->d_svel, sizeof(float4) * c->cap_spheres);
    ALLOC(c->d_pairA, sizeof(float4) * (c->cap_spheres / 2) * 4);      // A, B, U, V contiguous
    c->d_pairB = c->d_pairA + c->cap_spheres / 2;
    ALLOC(c->d_cost, sizeof(float) * 5 * max_agents);
    ALLOC(c->d_minclr, sizeof(float) * max_agents);
    ALLOC(c->d_collided, sizeof(int) * max_agents);
    ALLOC(c->d_vox_bitmap, sizeof(unsigned) * (1u << 20));
    ALLOC(c->d_vox_state, sizeof(unsigned long long) * 1024);
    ALLOC(c->d_vox_sync, sizeof(int) * 2);
    ALLOC(c->d_vox_count, sizeof(int));
    ALLOC(c->d_snap, sizeof(float) * 14 * max_agents);
    ALLOC(c->d_prev, sizeof(int));
    ALLOC(c->d_ap_rd, sizeof(float) * max_agents);
    ALLOC(c->d_ap_kf, sizeof(float) * max_agents);
    ALLOC(c->d_ap_idx, sizeof(int) * max_agents);
    ALLOC(c->d_sel_rec, sizeof(int) * 8);
    ALLOC(c->d_sel_ticket, sizeof(int));
    ALLOC(c->d_scratch, sizeof(float) * 64);
    ALLOC(c->d_sph_stats, sizeof(float) * 2);
#undef ALLOC
    if ((e = cudaMallocHost((void**)&c->h_pinned, sizeof(float) * hp)) != cudaSuccess ||
        (e = cudaMallocHost((void**)&c->h_best, sizeof(int) * 16)) != cudaSuccess ||
        (e = cudaMemset(c->d_sel_ticket, 0, sizeof(int))) != cudaSuccess ||
        (e = cudaMemset(c->d_vox_bitmap, 0, sizeof(unsigned) * (1u << 20))) != cudaSuccess ||
        (e = cudaMemset(c->d_vox_state, 0, sizeof(unsigned long long) * 1024)) != cudaSuccess ||
        (e = cudaMemset(c->d_vox_sync, 0, sizeof(int) * 2)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&c->ev_pinned, cudaEventDisableTiming)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&c->ev_ap, cudaEventDisableTiming)) != cudaSuccess ||
        (e = cudaMallocHost((void**)&c->h_ap, sizeof(float) * 3 * (size_t)max_agents)) != cudaSuccess ||
        (e = cudaEventCreate(&c->ev0)) != cudaSuccess || (e = cudaEventCreate(&c->ev1)) != cudaSuccess) {
        gmapp_destroy(c);
        return fail(nullptr, GMAPP_ECUDA, "pinned / event allocation: %s", cudaGetErrorString(e));
    }
    // opt every rollout variant in to the full dynamic shared memory of the device
    for (int kind = 0; kind < 2; ++kind)
        for (int at = 1; at <= (kind == 0 ? 2 : 1); ++at)
            for (int mv = 0; mv < 2; ++mv)
                for (int cu = 0; cu < 2; ++cu)
                    for (int st = 0; st < 2; ++st) {
                        e = cudaFuncSetAttribute((const void*)rollout_kernel(kind, at, mv, cu, st),
                                                 cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin);
                        if (e != cudaSuccess) { gmapp_destroy(c); return fail(nullptr, GMAPP_ECUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e)); }
                    }
    for (int mv = 0; mv < 2; ++mv)
        for (int cu = 0; cu < 8; ++cu) {
            e = cudaFuncSetAttribute((const void*)rollout_wide_kernel(mv, cu & 1, (cu >> 1) & 1, (cu >> 2) != 0),
                                     cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin);
            if (e != cudaSuccess) { gmapp_destroy(c); return fail(nullptr, GMAPP_ECUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e)); }
        }
    for (int at = 1; at <= 2; ++at)
        for (int md = 0; md < 5; ++md)
            for (int cu = 0; cu < 6; ++cu)
                for (int hf = 0; hf < 8; ++hf) {
                    const void* fn = (const void*)rollout_x2_kernel(at, md, cu & 1, cu >> 1, (hf & 1) != 0, (hf & 2) != 0, (hf & 4) != 0);
                    if (!fn) continue;                     // no such variant (tile ring with cull / sub-warp groups)
                    e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin);
                    if (e != cudaSuccess) { gmapp_destroy(c); return fail(nullptr, GMAPP_ECUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e)); }
                }
    *out = c;
    return GMAPP_OK;
}

extern "C" gmapp_status gmapp_destroy(gmapp_ctx* c) {
    if (!c) return GMAPP_OK;
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    cudaFree(c->d_sph_raw); cudaFree(c->d_sph_eff); cudaFree(c->d_svel); cudaFree(c->d_pairA);
    cudaFree(c->d_cost); cudaFree(c->d_minclr); cudaFree(c->d_collided);
    cudaFree(c->d_sel_rec); cudaFree(c->d_sel_ticket); cudaFree(c->d_scratch); cudaFree(c->d_sph_stats);
    cudaFree(c->d_ap_rd); cudaFree(c->d_ap_kf); cudaFree(c->d_ap_idx); cudaFree(c->d_snap); cudaFree(c->d_prev);
    cudaFree(c->d_vox_bitmap); cudaFree(c->d_vox_state); cudaFree(c->d_vox_sync); cudaFree(c->d_vox_count);
    if (c->h_ap) cudaFreeHost(c->h_ap);
    if (c->h_pinned) cudaFreeHost(c->h_pinned);
    if (c->h_best) cudaFreeHost(c->h_best);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    if (c->ev_pinned) cudaEventDestroy(c->ev_pinned);
    if (c->ev_ap) cudaEventDestroy(c->ev_ap);
    delete c;
    return GMAPP_OK;
}

extern "C" const char* gmapp_last_error(const gmapp_ctx* c) { return c ? c->err : g_create_err; }
extern "C" int gmapp_sm_count(const gmapp_ctx* c) { return c ? c->num_sms : 0; }

extern "C" gmapp_status gmapp_set_tuning(gmapp_ctx* c, const gmapp_tuning* t) {
    if (!c) return GMAPP_EINVAL;
    if (!t) { c->has_tuning = false; return GMAPP_OK; }
    if (t->lanes_per_agent < 0 || t->lanes_per_agent > 1024 ||
        (t->lanes_per_agent && (t->lanes_per_agent & (t->lanes_per_agent - 1))))
        return fail(c, GMAPP_EINVAL, "set_tuning: lanes_per_agent must be 0 or a power of two <= 1024%s");
    if (t->agents_per_thread < 0 || t->agents_per_thread > 2) return fail(c, GMAPP_EINVAL, "set_tuning: agents_per_thread must be 0, 1 or 2%s");
    if (t->cull < -1 || t->cull > 1 || t->stage < -1 || t->stage > 2 || t->max_ctas < 0 || t->scalar_path < 0 || t->scalar_path > 1)
        return fail(c, GMAPP_EINVAL, "set_tuning: cull in {-1,0,1}, stage in {-1,0,1,2}, max_ctas >= 0, scalar_path in {0,1}%s");
    c->tuning = *t; c->has_tuning = true;
    return GMAPP_OK;
}

extern "C" gmapp_status gmapp_get_launch_info(const gmapp_ctx* c, gmapp_launch_info* out) {
    if (!c || !out) return GMAPP_EINVAL;
    *out = c->info;
    return GMAPP_OK;
}

// ---------------------------------------------------------------------------------------------
// obstacles
// ---------------------------------------------------------------------------------------------
__global__ void k_set_int(int* p, int v) { *p = v; }

__global__ void k_add_ragent(const float4* __restrict__ raw, float4* __restrict__ eff, int n, int n_fill, float r_agent) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_fill) return;
    float4 s = raw[i];
    if (i < n) s.w += r_agent;
    eff[i] = s;
}

static int fill_count(const gmapp_ctx* c, int n) {
    int f = round_up(n > 0 ? n : 1, 2048);
    return f > c->cap_spheres ? c->cap_spheres : f;
}

static gmapp_status effective_pairs(gmapp_ctx* c, float r_agent, cudaStream_t st, int* launches);

extern "C" gmapp_status gmapp_set_obstacles(gmapp_ctx* c, const float* d_xyzr, const float* d_vel, int n, void* stream) {
    if (!c) return GMAPP_EINVAL;
    if (n < 0) return fail(c, GMAPP_EINVAL, "set_obstacles: n < 0%s");
    if (n > 0 && !d_xyzr) return fail(c, GMAPP_EINVAL, "set_obstacles: d_xyzr is NULL%s");
    if (n > c->max_spheres) return fail(c, GMAPP_ECAPACITY, "set_obstacles: n = %s%ld exceeds max_spheres = %ld", "", n, c->max_spheres);
    cudaStream_t st = (cudaStream_t)stream;
    const int nf = fill_count(c, n);
    // one launch: the float4 sphere array (+ velocities) and the sphere-pair arrays of the packed kernels for
    // r_agent = 0 (repacked lazily if a rollout asks for another r_agent)
    k_pack_spheres<<<(nf + 255) / 256, 256, 0, st>>>(d_xyzr, d_vel, n, nf, 0.0f, c->d_sph_raw, c->d_svel, c->d_pairA, c->cap_spheres / 2);
    CUDA_TRY(c, cudaGetLastError());
    c->n_spheres = n;
    c->built_world = false;
    c->moving = (d_vel != nullptr) && n > 0;
    c->eff_valid = false;
    c->pair_valid = true; c->pair_r_agent = 0.0f;
    c->stats_valid = false;
    return GMAPP_OK;
}

// ---------------------------------------------------------------------------------------------
// sphere-world builder (NEXT row N3): point cloud -> crop -> voxelise -> occupied-voxel centres as S_W, on the device
// ---------------------------------------------------------------------------------------------
extern "C" gmapp_status gmapp_build_sphere_world(gmapp_ctx* c, const float* d_points, int n_points, const float* lo,
                                                 const float* hi, float pitch, int capacity, int32_t* d_count_out,
                                                 void* stream) {
    if (!c) return GMAPP_EINVAL;
    if (n_points < 0 || (n_points > 0 && !d_points) || !lo || !hi) return fail(c, GMAPP_EINVAL, "build_sphere_world: NULL points / bounds or n_points < 0%s");
    if (!isfinite(pitch) || !(pitch > 0.0f)) return fail(c, GMAPP_EINVAL, "build_sphere_world: pitch must be finite and > 0%s");
    if (capacity < 1) return fail(c, GMAPP_EINVAL, "build_sphere_world: capacity must be >= 1%s");
    if (capacity > c->max_spheres) return fail(c, GMAPP_ECAPACITY, "build_sphere_world: capacity = %s%ld exceeds max_spheres = %ld", "", capacity, c->max_spheres);
    VoxelGrid G;
    double nvox = 1.0;
    for (int a = 0; a < 3; ++a) {
        if (!isfinite(lo[a]) || !isfinite(hi[a]) || !(hi[a] > lo[a])) return fail(c, GMAPP_EINVAL, "build_sphere_world: need finite lo < hi%s");
        G.lo[a] = lo[a]; G.hi[a] = hi[a];
        const double d = ceil(((double)hi[a] - (double)lo[a]) / (double)pitch);
        if (d > 4096.0) return fail(c, GMAPP_ECAPACITY, "build_sphere_world: more than 4096 voxels along an axis%s");
        G.dim[a] = d < 1.0 ? 1 : (int)d;
        nvox *= G.dim[a];
    }
    if (nvox > (double)(1u << 25)) return fail(c, GMAPP_ECAPACITY, "build_sphere_world: the voxel grid exceeds 2^25 voxels%s");
    G.pitch = pitch;
    G.n_words = ((int)nvox + 31) / 32;
    const int n_blocks = (G.n_words + 1023) / 1024;
    cudaStream_t st = (cudaStream_t)stream;
    const int nf = fill_count(c, capacity);
    if (G.n_words <= kVoxSmallWords) {
        // small grids (the paper's workspace): ONE launch -- per-block bitmaps in shared memory, merged, and the block that
        // finishes last scans and emits (gmapp_voxel.cuh)
        int grid = (n_points + 2047) / 2048;                // two points per thread
        if (grid < 1) grid = 1;
        if (grid > 2 * c->num_sms) grid = 2 * c->num_sms;
        k_vox_build_small<<<grid, 1024, sizeof(unsigned) * G.n_words, st>>>(d_points, n_points, G, c->d_vox_bitmap, c->d_vox_sync, capacity, nf,
                                                                       c->d_sph_raw, c->d_svel, c->d_pairA, c->cap_spheres / 2,
                                                                       c->d_vox_count, d_count_out);
        CUDA_TRY(c, cudaGetLastError());
        c->n_spheres = capacity; c->built_world = true; c->moving = false; c->eff_valid = false;
        c->pair_valid = true; c->pair_r_agent = 0.0f; c->stats_valid = false;
        return GMAPP_OK;
    }
    // large grids, two launches: mark the global bitmap (it is zero: every build leaves it so), then ONE kernel that scans,
    // emits the spheres into the float4 array and the sphere-pair arrays (r_agent = 0), writes the sentinel tail and the
    // count, and zeroes the bitmap and its own scan state again
    if (n_points > 0) k_vox_mark<<<(n_points + 255) / 256, 256, 0, st>>>(d_points, n_points, G, c->d_vox_bitmap);
    int n_help = (nf + 1023) / 1024;                       // fill helpers: the sentinel tail in parallel
    if (n_help > 64) n_help = 64;
    k_vox_compact<<<n_blocks + n_help, 1024, 0, st>>>(c->d_vox_bitmap, c->d_vox_state, c->d_vox_sync, G, capacity, nf, n_blocks,
                                                      c->d_sph_raw, c->d_svel, c->d_pairA, c->cap_spheres / 2, c->d_vox_count, d_count_out);
    CUDA_TRY(c, cudaGetLastError());
    // the sphere world now holds `capacity` slots: the occupied voxels first, sentinels behind them
    c->n_spheres = capacity;
    c->built_world = true;
    c->moving = false;
    c->eff_valid = false;
    c->pair_valid = true; c->pair_r_agent = 0.0f;
    c->stats_valid = false;
    return GMAPP_OK;
}

extern "C" gmapp_status gmapp_get_obstacles(gmapp_ctx* c, float* d_xyzr_out, int n, void* stream) {
    if (!c) return GMAPP_EINVAL;
    if (c->n_spheres < 0) return fail(c, GMAPP_ESTATE, "get_obstacles: no sphere world has been set%s");
    if (n < 0 || n > c->n_spheres || (n > 0 && !d_xyzr_out)) return fail(c, GMAPP_EINVAL, "get_obstacles: need 0 <= n <= %s%ld spheres and a buffer", "", c->n_spheres);
    if (n > 0) CUDA_TRY(c, cudaMemcpyAsync(d_xyzr_out, c->d_sph_raw, sizeof(float4) * (size_t)n, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return GMAPP_OK;
}

extern "C" gmapp_status gmapp_set_obstacles_host(gmapp_ctx* c, const float* h_xyzr, const float* h_vel, int n, void* stream) {
    if (!c) return GMAPP_EINVAL;
    if (n < 0) return fail(c, GMAPP_EINVAL, "set_obstacles_host: n < 0%s");
    if (n > 0 && !h_xyzr) return fail(c, GMAPP_EINVAL, "set_obstacles_host: h_xyzr is NULL%s");
    if (n > c->max_spheres) return fail(c, GMAPP_ECAPACITY, "set_obstacles_host: n = %s%ld exceeds max_spheres = %ld", "", n, c->max_spheres);
    cudaStream_t st = (cudaStream_t)stream;
    if (n > 0) {
        // the pinned buffer may still be read by the packing kernel of an earlier host call -- on ANY stream: wait for
        // the event recorded behind that kernel
        if (c->pinned_busy) { CUDA_TRY(c, cudaEventSynchronize(c->ev_pinned)); c->pinned_busy = false; }
        memcpy(c->h_pinned, h_xyzr, sizeof(float) * 4 * n);
        if (h_vel) memcpy(c->h_pinned + 4 * (size_t)n, h_vel, sizeof(float) * 3 * n);
    }
    // the packing kernel reads the pinned host buffer itself (unified addressing: one read over the host link instead
    // of a copy-engine transfer into a staging buffer followed by the same read)
    gmapp_status s = gmapp_set_obstacles(c, c->h_pinned, h_vel ? c->h_pinned + 4 * (size_t)n : nullptr, n, stream);
    if (s == GMAPP_OK && n > 0) { CUDA_TRY(c, cudaEventRecord(c->ev_pinned, st)); c->pinned_busy = true; }
    return s;
}

// sphere array with R = r + r_agent; launches the tiny repack kernel only when r_agent changed
static gmapp_status effective_spheres(gmapp_ctx* c, float r_agent, cudaStream_t st, const float4** out, int* launches) {
    if (r_agent == 0.0f) { *out = c->d_sph_raw; return GMAPP_OK; }
    if (!c->eff_valid || c->eff_r_agent != r_agent) {
        const int nf = fill_count(c, c->n_spheres);
        k_add_ragent<<<(nf + 255) / 256, 256, 0, st>>>(c->d_sph_raw, c->d_sph_eff, c->n_spheres, nf, r_agent);
        CUDA_TRY(c, cudaGetLastError());
        c->eff_valid = true; c->eff_r_agent = r_agent;
        if (launches) ++*launches;
    }
    *out = c->d_sph_eff;
    return GMAPP_OK;
}

// sphere-pair arrays with R = r + r_agent; launches the tiny repack kernel only when spheres or r_agent changed
static gmapp_status effective_pairs(gmapp_ctx* c, float r_agent, cudaStream_t st, int* launches) {
    if (c->pair_valid && c->pair_r_agent == r_agent) return GMAPP_OK;
    const int n2f = fill_count(c, c->n_spheres) / 2;
    k_pack_pairs<<<(n2f + 255) / 256, 256, 0, st>>>(c->d_sph_raw, c->moving ? c->d_svel : nullptr, c->n_spheres, n2f, r_agent,
                                                    c->d_pairA, c->cap_spheres / 2);
    CUDA_TRY(c, cudaGetLastError());
    c->pair_valid = true; c->pair_r_agent = r_agent;
    c->stats_valid = false;
    if (launches) ++*launches;
    return GMAPP_OK;
}

// {largest R, largest sphere speed} of the current pair arrays, for the tile ring's refinement prediction; one small
// launch per sphere world (only when a rollout takes the ring)
__global__ void __launch_bounds__(1024) k_sphere_stats(const float4* __restrict__ pairs, int stride, int n2, int moving, float* out) {
    float rmax = 0.0f, u2max = 0.0f;
    for (int j = threadIdx.x; j < n2; j += blockDim.x) {
        const float4 b = pairs[stride + j];
        rmax = fmaxf(rmax, fmaxf(-b.z, -b.w));
        if (moving) {
            const float4 u = pairs[2 * stride + j], w = pairs[3 * stride + j];
            u2max = fmaxf(u2max, fmaxf(fmaf(u.x, u.x, fmaf(u.z, u.z, w.x * w.x)), fmaf(u.y, u.y, fmaf(u.w, u.w, w.y * w.y))));
        }
    }
    __shared__ float sr[32], su[32];
    for (int off = 16; off > 0; off >>= 1) {
        rmax = fmaxf(rmax, __shfl_xor_sync(0xffffffffu, rmax, off));
        u2max = fmaxf(u2max, __shfl_xor_sync(0xffffffffu, u2max, off));
    }
    if ((threadIdx.x & 31) == 0) { sr[threadIdx.x >> 5] = rmax; su[threadIdx.x >> 5] = u2max; }
    __syncthreads();
    if (threadIdx.x < 32) {
        rmax = sr[threadIdx.x]; u2max = su[threadIdx.x];
        for (int off = 16; off > 0; off >>= 1) {
            rmax = fmaxf(rmax, __shfl_xor_sync(0xffffffffu, rmax, off));
            u2max = fmaxf(u2max, __shfl_xor_sync(0xffffffffu, u2max, off));
        }
        if (threadIdx.x == 0) { out[0] = rmax; out[1] = sqrtf(u2max) * 1.000001f; }
    }
}
static gmapp_status sphere_stats(gmapp_ctx* c, cudaStream_t st, int* launches) {
    if (c->stats_valid) return GMAPP_OK;
    k_sphere_stats<<<1, 1024, 0, st>>>(c->d_pairA, c->cap_spheres / 2, fill_count(c, c->n_spheres) / 2, c->moving ? 1 : 0, c->d_sph_stats);
    CUDA_TRY(c, cudaGetLastError());
    c->stats_valid = true;
    if (launches) ++*launches;
    return GMAPP_OK;
}

static gmapp_status check_gains(gmapp_ctx* c, const gmapp_gains* g, const char* who) {
    if (!g) return fail(c, GMAPP_EINVAL, "%s: gains is NULL", who);
    const float* f = &g->k_circ;
    for (int i = 0; i < 18; ++i) if (!isfinite(f[i])) return fail(c, GMAPP_EINVAL, "%s: non-finite gain", who);
    if (!(g->eps_dist > 0.0f) || !(g->r_influence > 0.0f) || g->eps_dist > g->r_influence)
        return fail(c, GMAPP_EINVAL, "%s: need 0 < eps_dist <= r_influence (Alg. 1 lines 6-7)", who);
    if (g->r_agent < 0.0f || g->r_cost_goal < 0.0f || g->r_cost_obs < 0.0f || !(g->a_max > 0.0f))
        return fail(c, GMAPP_EINVAL, "%s: r_agent, r_cost_* must be >= 0 and a_max > 0", who);
    if (g->heuristic != 0 && g->heuristic != 1) return fail(c, GMAPP_EINVAL, "%s: heuristic must be 0 (circular field / MFI, Eq. 2-3) or 1 (APF, Eq. 1)", who);
    return GMAPP_OK;
}

// ---------------------------------------------------------------------------------------------
// heterogeneous ensemble: per-agent detection radius, gain and heuristic
// ---------------------------------------------------------------------------------------------
extern "C" gmapp_status gmapp_set_agent_params(gmapp_ctx* c, const float* h_r_influence, const float* h_k_circ,
                                               const int32_t* h_heuristic, int n, void* stream) {
    if (!c) return GMAPP_EINVAL;
    if (n < 0) return fail(c, GMAPP_EINVAL, "set_agent_params: n < 0%s");
    if (n > c->max_agents) return fail(c, GMAPP_ECAPACITY, "set_agent_params: n = %s%ld exceeds max_agents = %ld", "", n, c->max_agents);
    if (n == 0 || (!h_r_influence && !h_k_circ && !h_heuristic)) { c->ap_n = 0; return GMAPP_OK; }
    float min_rd = INFINITY;
    for (int i = 0; i < n; ++i) {
        if (h_r_influence) {
            if (!isfinite(h_r_influence[i]) || !(h_r_influence[i] > 0.0f)) return fail(c, GMAPP_EINVAL, "set_agent_params: r_influence[%s%ld] must be finite and > 0", "", i);
            if (h_r_influence[i] < min_rd) min_rd = h_r_influence[i];
        }
        if (h_k_circ && !isfinite(h_k_circ[i])) return fail(c, GMAPP_EINVAL, "set_agent_params: k_circ[%s%ld] is not finite", "", i);
        if (h_heuristic && h_heuristic[i] != 0 && h_heuristic[i] != 1) return fail(c, GMAPP_EINVAL, "set_agent_params: heuristic[%s%ld] must be 0 or 1", "", i);
    }
    cudaStream_t st = (cudaStream_t)stream;
    // the pinned staging may still be in flight from an earlier call -- on any stream: wait for the event behind its copies
    if (c->ap_busy) { CUDA_TRY(c, cudaEventSynchronize(c->ev_ap)); c->ap_busy = false; }
    float* hrd = c->h_ap; float* hkf = c->h_ap + c->max_agents; int* hidx = (int*)(c->h_ap + 2 * (size_t)c->max_agents);
    c->ap_count[0] = c->ap_count[1] = 0;
    if (h_heuristic) {                               // stable grouping: circular-field agents first, then APF agents
        int k = 0;
        for (int h = 0; h < 2; ++h)
            for (int i = 0; i < n; ++i) if (h_heuristic[i] == h) { hidx[k++] = i; ++c->ap_count[h]; }
        CUDA_TRY(c, cudaMemcpyAsync(c->d_ap_idx, hidx, sizeof(int) * n, cudaMemcpyHostToDevice, st));
    }
    if (h_r_influence) {
        memcpy(hrd, h_r_influence, sizeof(float) * n);
        CUDA_TRY(c, cudaMemcpyAsync(c->d_ap_rd, hrd, sizeof(float) * n, cudaMemcpyHostToDevice, st));
    }
    if (h_k_circ) {
        memcpy(hkf, h_k_circ, sizeof(float) * n);
        CUDA_TRY(c, cudaMemcpyAsync(c->d_ap_kf, hkf, sizeof(float) * n, cudaMemcpyHostToDevice, st));
    }
    CUDA_TRY(c, cudaEventRecord(c->ev_ap, st)); c->ap_busy = true;
    c->ap_n = n; c->ap_has_rd = h_r_influence != nullptr; c->ap_has_kf = h_k_circ != nullptr; c->ap_has_h = h_heuristic != nullptr;
    c->ap_min_rd = min_rd;
    return GMAPP_OK;
}

// ---------------------------------------------------------------------------------------------
// launch selection
// ---------------------------------------------------------------------------------------------
struct LaunchCfg { int at, L, groups, block, grid, agents_per_cta, stage, cull, n_pad, smem, tile_off, red_off; };

static gmapp_status choose_launch(gmapp_ctx* c, int kind, int n_agents, LaunchCfg* o) {
    const gmapp_tuning* t = c->has_tuning ? &c->tuning : nullptr;
    int max_ctas = c->num_sms;
    if (t && t->max_ctas > 0 && t->max_ctas < max_ctas) max_ctas = t->max_ctas;
    const int A = (n_agents + max_ctas - 1) / max_ctas;
    const int grid = (n_agents + A - 1) / A;
    int at = (kind == GMAPP_POINT3 && A >= 2) ? 2 : 1;
    if (t && t->agents_per_thread) at = t->agents_per_thread;
    if (kind == GMAPP_MOTOR6) at = 1;
    const int G = (A + at - 1) / at;
    const int tmax = rollout_max_threads(kind, at);
    if (G > tmax) return fail(c, GMAPP_ECAPACITY, "rollout: %s%ld agent groups per CTA exceed %ld threads", "", G, tmax);
    const int ns = c->n_spheres;
    int L;
    if (t && t->lanes_per_agent) {
        L = t->lanes_per_agent;
        if (G * L > tmax) return fail(c, GMAPP_EINVAL, "rollout: lanes_per_agent %s%ld x %ld groups exceeds the thread limit", "", L, G);
    } else {
        L = pow2_floor(tmax / G);
        const int cap = pow2_ceil(ns > 0 ? ns : 1);       // no more lanes than spheres
        if (L > cap) L = cap;
    }
    if (L > 32 && G > kMaxGroupsNamedBar) {
        if (t && t->lanes_per_agent) return fail(c, GMAPP_EINVAL, "rollout: lanes_per_agent > 32 allows at most 15 groups per CTA, need %s%ld", "", G);
        L = 32;
    }
    o->at = at; o->L = L; o->groups = G; o->grid = grid; o->agents_per_cta = A;
    o->block = round_up(G * L, 32);
    o->n_pad = ns > 0 ? round_up(ns, L) : 0;
    o->cull = (t && t->cull >= 0) ? t->cull : 0;
    // dynamic shared memory: [0,64) mbarrier; [64, 64+2 KB) cross-warp exchange; then the sphere tile
    o->red_off = 64;
    o->tile_off = 64 + 2 * 32 * 2 * 16;
    const size_t tile_bytes = (size_t)o->n_pad * 16 * (c->moving ? 2 : 1);
    const bool fits = o->tile_off + tile_bytes <= (size_t)c->smem_optin;
    int stage = fits ? 1 : 0;
    if (t && t->stage >= 0) {
        if (t->stage == 1 && !fits) return fail(c, GMAPP_EINVAL, "rollout: sphere set (%s%ld bytes) does not fit shared memory", "", (long)tile_bytes);
        if (t->stage <= 1) stage = t->stage;             // the tile ring (2) belongs to the packed kernels; here: automatic
    }
    if (o->n_pad == 0) stage = 0;
    o->stage = stage;
    o->smem = o->tile_off + (stage == 1 ? (int)tile_bytes : 0);
    return GMAPP_OK;
}


// ---------------------------------------------------------------------------------------------
// packed f32x2 rollout (POINT3, static or moving spheres): launch selection + launch
// ---------------------------------------------------------------------------------------------
struct X2Plan { int Lk, A, grid, at, G, L, mode, n2p, cull, stage, ring_tp, xch_off, rec_off, tile_off, pair_bytes, block, smem; size_t tile_bytes; };

// launch selection alone (no CUDA call): every reason to refuse a launch shape is found here, before anything is enqueued
static gmapp_status plan_rollout_x2(gmapp_ctx* c, int n_agents, X2Plan* o) {
    const gmapp_tuning* t = c->has_tuning ? &c->tuning : nullptr;
    int max_ctas = c->num_sms;
    if (t && t->max_ctas > 0 && t->max_ctas < max_ctas) max_ctas = t->max_ctas;
    int A = (n_agents + max_ctas - 1) / max_ctas;                 // agents per CTA: one wave of the SMs
    if (A > 1024) A = 1024;                                       // beyond 1024 agents per CTA: several waves of CTAs
    const int grid = (n_agents + A - 1) / A;
    int at = A >= 2 ? 2 : 1;
    if (t && t->agents_per_thread) at = t->agents_per_thread;
    int G = (A + at - 1) / at;                                    // groups per CTA
    // 9 to 16 one-warp groups: round the warp count up to a multiple of 4 (the kernel then gives the first A - G warps
    // two agents and the others one), so that the four schedulers of an SM carry the same number of agent-sweeps
    if (at == 2 && G >= 9 && G <= 16 && !(t && t->lanes_per_agent)) G = (G + 3) & ~3;
    const int tmax = kX2SweepThreads;
    const int ns = c->n_spheres;
    const int n2 = (ns + 1) / 2;
    // more than two agents per warp: every warp walks a block of agents in chunks of two (mode 4)
    const bool chunked = A > 32 && n2 >= 32 && at == 2 && !(t && t->lanes_per_agent && t->lanes_per_agent != 32);
    if (chunked && A > 1024) return fail(c, GMAPP_ECAPACITY, "rollout: %s%ld agents per CTA exceed the 1024 state records", "", A);
    if (!chunked && G > tmax) return fail(c, GMAPP_ECAPACITY, "rollout: %s%ld agent groups per CTA exceed %ld threads", "", G, tmax);
    int L;
    if (chunked) {
        L = 32; G = tmax / 32;
    } else if (t && t->lanes_per_agent) {
        L = t->lanes_per_agent;
        if (G * L > tmax) return fail(c, GMAPP_EINVAL, "rollout: lanes_per_agent %s%ld x %ld groups exceeds the thread limit", "", L, G);
        if (L > 32 && G > 7) return fail(c, GMAPP_EINVAL, "rollout: lanes_per_agent > 32 allows at most 7 groups per CTA, need %s%ld", "", G);
    } else {
        L = pow2_floor(tmax / G);
        int cap = pow2_ceil(n2 > 0 ? n2 : 1);                     // no more lanes than sphere pairs ...
        if (cap < 32 && n2 > 0) cap = 32;                         // ... but a whole warp per group when it fits: the full-warp
        if (L > cap) L = cap;                                     // reduction beats the sub-warp one even with idle lanes
        if (L > 32 && G > 7) L = 32;                              // two named barriers per multi-warp group
    }
    // 5 to 7 two-agent groups per CTA: mixed group widths -- 16 sweep warps, the first 2 G - 8 groups 64 lanes wide, the others
    // 128, one epilogue warp per two groups (gmapp_rollout_x2.cuh, group_epilogue_warp2); needs at least 128 sphere pairs
    if (!chunked && at == 2 && L >= 64 && G >= 5 && G <= 7 && pow2_ceil(n2 > 0 ? n2 : 1) < 128) L = 32;
    const int mode = chunked ? 4 : (L >= 64 ? (G <= 4 ? 2 : 3) : (L == 32 ? 1 : 0));
    const bool mixed = mode == 3 && at == 2;
    if (mixed && L != 64) return fail(c, GMAPP_EINVAL, "rollout: 5 to 7 two-agent groups per CTA take lanes_per_agent = 64 (mixed 64 / 128), got %s%ld", "", L);
    const int Lk = mixed ? 128 : L;                               // what the kernel pads the pair arrays to (P.L)
    const int n2p = n2 > 0 ? round_up(n2, Lk) : 0;
    const int cull = (t && t->cull >= 0) ? t->cull : 0;
    // dynamic shared memory: [0,64) mbarriers; then the exchange area of the multi-warp groups (per group: the
    // per-lane partials of two agents + the published states = (2 L + 8) float4) or, mode 4, the 24-word state
    // record of every agent; then the sphere-pair tile
    const int xch_off = 64, rec_off = 128;
    const int tile_off = rec_off + (chunked ? round_up(A * 24 * 4, 128)
                                            : mixed ? round_up(((2 * G - 8) * 136 + (8 - G) * 264) * 16, 128)
                                            : (mode >= 2 ? round_up(G * (2 * L + 8) * 16, 128) : 0));
    const int pair_bytes = c->moving ? 64 : 32;                          // pair arrays A, B (+ U, V when the spheres move)
    const size_t tile_bytes = (size_t)n2p * pair_bytes;
    const bool fits = tile_off + tile_bytes <= (size_t)c->smem_optin;
    // sets beyond shared memory: a ring of kRingStages tiles fed by TMA bulk copies (stage 2); the branch-free kernels of
    // modes 1, 2, 4 have it, the warp-vote variant and sub-warp groups read through L1 / L2 (stage 0)
    const bool ring_ok = mode != 0 && cull == 0;
    int ring_tp = 0;
    if (ring_ok) {
        ring_tp = pow2_floor((int)(((size_t)c->smem_optin - tile_off) / ((size_t)kRingStages * pair_bytes)));
        if (ring_tp > 2048) ring_tp = 2048;
        if (ring_tp < Lk) ring_tp = 0;                                   // a tile must hold a whole trip of the group
    }
    // Measured on B200 at equal sphere density (profiles/r02_tile_ring.md): the ring beats the L1/L2 path by 3-5 % once the set is
    // far beyond L1 (>= 8 tiles, i.e. 32768 static spheres) for one-warp groups and chunked warps; at 4 tiles the two are level, and
    // with multi-warp groups (16 trips per tile and warp) the per-tile hand-over costs more than L1 misses do.
    const int ring_tiles = ring_tp > 0 ? (n2p + ring_tp - 1) / ring_tp : 0;
    const bool ring_wins = ring_tiles >= 8 && (mode == 1 || mode == 4);
    int stage = fits ? 1 : (ring_wins ? 2 : 0);
    if (t && t->stage >= 0) {
        if (t->stage == 1 && !fits) return fail(c, GMAPP_EINVAL, "rollout: sphere set (%s%ld bytes) does not fit shared memory", "", (long)tile_bytes);
        if (t->stage == 2 && ring_tp == 0) return fail(c, GMAPP_EINVAL, "rollout: the tile ring needs the branch-free kernel and whole-warp groups%s");
        stage = t->stage;
    }
    if (n2p == 0) stage = 0;
    o->A = A; o->grid = grid; o->at = at; o->G = G; o->L = L; o->mode = mode; o->n2p = n2p; o->cull = cull; o->stage = stage;
    o->ring_tp = ring_tp; o->xch_off = xch_off; o->rec_off = rec_off; o->tile_off = tile_off; o->pair_bytes = pair_bytes;
    o->tile_bytes = tile_bytes;
    // mixed widths: 16 sweep warps + one epilogue warp per TWO groups (kernel table: MAXT 576 is the tag of that variant)
    o->block = mode == 4 ? tmax : (mixed ? 32 * (16 + (G + 1) / 2) : (mode >= 2 ? G * L + 32 * G : round_up(G * L, 32)));
    o->Lk = Lk;
    o->smem = tile_off + (stage == 1 ? (int)tile_bytes : (stage == 2 ? kRingStages * ring_tp * pair_bytes : 0));
    return GMAPP_OK;
}

static gmapp_status launch_rollout_x2(gmapp_ctx* c, const float* d_agents, float* d_agents_out, int n_agents,
                                      const float* goal, const gmapp_gains* g, float dt, int steps, cudaStream_t st) {
    X2Plan pl;
    gmapp_status s = plan_rollout_x2(c, n_agents, &pl);
    if (s != GMAPP_OK) return s;
    const int A = pl.A, grid = pl.grid, at = pl.at, L = pl.L, mode = pl.mode, n2p = pl.n2p, cull = pl.cull, stage = pl.stage;
    const int ring_tp = pl.ring_tp, xch_off = pl.xch_off, rec_off = pl.rec_off, tile_off = pl.tile_off, block = pl.block, smem = pl.smem;
    int launches = 0;
    s = effective_pairs(c, g->r_agent, st, &launches);
    if (s != GMAPP_OK) return s;
    if (stage == 2 && c->moving) {                                       // largest sphere speed, for the ring's refinement prediction
        s = sphere_stats(c, st, &launches);
        if (s != GMAPP_OK) return s;
    }
    RolloutX2Params P;
    memset(&P, 0, sizeof P);
    P.pairA = c->d_pairA; P.pairB = c->d_pairB; P.n2p = n2p;
    P.agents_in = d_agents; P.agents_out = d_agents_out;
    P.n_agents = n_agents; P.agents_per_cta = A;
    P.L = pl.Lk; P.logL = ilog2(pl.Lk);
    P.steps = steps;
    for (int i = 0; i < 3; ++i) P.goal[i] = goal[i];
    P.dt = dt; P.t0 = c->roll_t0;
    P.k_circ = g->k_circ; P.k_att = g->k_att; P.k_damp = g->k_damp;
    P.c_lin = g->vel_factor * dt * g->inv_mass;
    P.inv_mass = g->inv_mass; P.vel_factor = g->vel_factor;
    P.r_d = g->r_influence; P.eps = g->eps_dist;
    P.apf = g->heuristic == 1;
    P.rcg = g->r_cost_goal > 0.0f ? g->r_cost_goal : g->r_influence;
    P.rco = g->r_cost_obs > 0.0f ? g->r_cost_obs : g->r_influence;
    P.rcg_is_rd = !(g->r_cost_goal > 0.0f); P.rco_is_rd = !(g->r_cost_obs > 0.0f);
    P.w_goal = g->w_goal; P.w_obs = g->w_obs; P.w_path = g->w_path; P.w_smooth = g->w_smooth; P.a_max = g->a_max;
    P.cost = c->d_cost; P.minclr = c->d_minclr; P.collided = c->d_collided;
    P.agent_idx = c->sub_idx;
    P.snap_out = c->roll_snap; P.snap_step = c->roll_snap_step; P.traj_out = c->roll_traj;
    P.count_dev = c->built_world ? c->d_vox_count : nullptr; P.n_cap = c->n_spheres;
    P.rd_arr = (c->ap_n > 0 && c->ap_has_rd) ? c->d_ap_rd : nullptr;
    P.kf_arr = (c->ap_n > 0 && c->ap_has_kf) ? c->d_ap_kf : nullptr;
    P.tile_off = tile_off; P.xch_off = xch_off; P.rec_off = rec_off;
    P.ring_tp = ring_tp; P.ring_off = 16; P.sph_stats = c->d_sph_stats;
    if (c->sel_want && GMAPP_FUSED_SELECT_X2) {           // selection fused into the tail of this launch (off by default: gmapp_kernels.cuh)
        P.sel.ticket = c->d_sel_ticket; P.sel.total = c->sel_total; P.sel.alpha = c->sel_alpha; P.sel.prev = c->sel_prev;
        P.sel.prev_dev = c->sel_prev_dev; P.sel.out_dev = c->d_sel_rec; P.sel.out_host = c->h_best; P.sel.seq = c->sel_seq;
        c->sel_fused = true;
    }
    P.stage = stage;
    rollout_x2_fn fn = rollout_x2_kernel(at, mode, cull != 0, stage, g->heuristic == 1, P.snap_out != nullptr || P.traj_out != nullptr, c->moving);
    fn<<<grid, block, smem, st>>>(P);
    CUDA_TRY(c, cudaGetLastError());
    ++launches;
    c->last_n_agents = n_agents;
    gmapp_launch_info& I = c->info;
    I.grid = grid; I.block = block; I.lanes_per_agent = L; I.agents_per_thread = at;
    I.agents_per_cta = A; I.cull = cull; I.stage = stage;
    I.tile_spheres = stage == 1 ? 2 * n2p : (stage == 2 ? 2 * ring_tp : 0);
    I.n_tiles = stage == 1 ? 1 : (stage == 2 ? (n2p + ring_tp - 1) / ring_tp : 0);
    I.smem_bytes = smem; I.kernels_launched = launches; I.packed_x2 = 1;
    cudaFuncAttributes fa;
    if (cudaFuncGetAttributes(&fa, (const void*)fn) == cudaSuccess) I.regs_per_thread = fa.numRegs;
    return GMAPP_OK;
}

// ---------------------------------------------------------------------------------------------
// rollout
// ---------------------------------------------------------------------------------------------
static gmapp_status rollout_sub(gmapp_ctx* c, gmapp_kind kind, const float* d_agents, float* d_agents_out, int n_agents,
                                const float* goal, const gmapp_gains* g, float dt, int steps, cudaStream_t stream);

// dry run of the launch selection of every launch this rollout will issue: refuses before anything is enqueued
static gmapp_status check_launchable(gmapp_ctx* c, gmapp_kind kind, int n_agents) {
    int counts[2] = {n_agents, 0};
    if (c->ap_n > 0 && c->ap_has_h) { counts[0] = c->ap_count[0]; counts[1] = c->ap_count[1]; }
    for (int h = 0; h < 2; ++h) {
        if (counts[h] <= 0) continue;
        gmapp_status s;
        if (kind == GMAPP_POINT3 && !(c->has_tuning && c->tuning.scalar_path)) { X2Plan pl; s = plan_rollout_x2(c, counts[h], &pl); }
        else { LaunchCfg cfg; s = choose_launch(c, kind, counts[h], &cfg); }
        if (s != GMAPP_OK) return s;
    }
    return GMAPP_OK;
}

extern "C" gmapp_status gmapp_rollout(gmapp_ctx* c, gmapp_kind kind, const float* d_agents, float* d_agents_out,
                                      int n_agents, const float* goal, const gmapp_gains* g, float dt, int steps,
                                      void* stream) {
    if (!c) return GMAPP_EINVAL;
    if (kind != GMAPP_POINT3 && kind != GMAPP_MOTOR6) return fail(c, GMAPP_EINVAL, "rollout: unknown kind%s");
    if (!d_agents || !goal) return fail(c, GMAPP_EINVAL, "rollout: NULL agents or goal%s");
    if (n_agents < 1 || steps < 1) return fail(c, GMAPP_EINVAL, "rollout: n_agents and steps must be >= 1%s");
    if (!isfinite(dt) || !(dt > 0.0f)) return fail(c, GMAPP_EINVAL, "rollout: dt must be finite and > 0%s");
    if (n_agents > c->max_agents) return fail(c, GMAPP_ECAPACITY, "rollout: n_agents = %s%ld exceeds max_agents = %ld", "", n_agents, c->max_agents);
    if (c->n_spheres < 0) return fail(c, GMAPP_ESTATE, "rollout: gmapp_set_obstacles has not been called%s");
    gmapp_status s = check_gains(c, g, "rollout");
    if (s != GMAPP_OK) return s;
    const int ng = kind == GMAPP_POINT3 ? 3 : 8;
    for (int i = 0; i < ng; ++i) if (!isfinite(goal[i])) return fail(c, GMAPP_EINVAL, "rollout: non-finite goal%s");
    c->sub_idx = nullptr;
    if (c->ap_n > 0) {                      // every check comes before the first enqueue: on error nothing is launched
        if (c->ap_n != n_agents) return fail(c, GMAPP_EINVAL, "rollout: gmapp_set_agent_params was given %s%ld agents, the rollout %ld", "", c->ap_n, n_agents);
        if (c->ap_has_rd && g->eps_dist > c->ap_min_rd) return fail(c, GMAPP_EINVAL, "rollout: need eps_dist <= every per-agent r_influence%s");
    }
    {   // launch shapes that cannot run are refused here too (a dry run of the launch selection)
        s = check_launchable(c, kind, n_agents);
        if (s != GMAPP_OK) return s;
    }
    if (c->roll_traj) {                     // pose 0 of every path = the start state, as given
        const size_t wb = sizeof(float) * (kind == GMAPP_POINT3 ? 6 : 14);
        CUDA_TRY(c, cudaMemcpy2DAsync(c->roll_traj, wb * (size_t)(steps + 1), d_agents, wb, wb, (size_t)n_agents,
                                      cudaMemcpyDefault, (cudaStream_t)stream));
    }
    // Selection fused into the rollout's tail: the packed kernels (every POINT3 launch, also one per heuristic) and the
    // wide 6D kernel (single launch) have it; after the scalar kernel gmapp_best_agent launches the selection kernel.
    c->sel_fused = false;
    c->sel_total = n_agents;
    c->sel_seq = (c->sel_seq % 0x3fffffff) + 1;
    c->sel_want = !(c->has_tuning && c->tuning.scalar_path) && (kind == GMAPP_POINT3 || !(c->ap_n > 0 && c->ap_has_h));
    c->fused_alpha = c->sel_alpha; c->fused_prev = c->sel_prev; c->fused_prev_dev = c->sel_prev_dev != nullptr;
    if (c->ap_n > 0) {
        // heterogeneous ensemble: one launch per heuristic over that heuristic's agents (the paper runs one
        // specialised kernel per heuristic), per-agent r_d / k_f read inside the kernels
        if (c->ap_has_h) {
            int total = 0;
            gmapp_launch_info first; memset(&first, 0, sizeof first);
            const int* idx = c->d_ap_idx;
            for (int h = 0; h < 2; ++h) {
                const int nh = c->ap_count[h];
                if (nh > 0) {
                    gmapp_gains gh = *g; gh.heuristic = h;
                    c->sub_idx = idx;
                    s = rollout_sub(c, kind, d_agents, d_agents_out, nh, goal, &gh, dt, steps, (cudaStream_t)stream);
                    c->sub_idx = nullptr;
                    if (s != GMAPP_OK) return s;
                    total += c->info.kernels_launched;
                }
                idx += nh;
            }
            c->info.kernels_launched = total;
            c->info.selection_fused = c->sel_fused ? 1 : 0;
            c->last_n_agents = n_agents;
            return GMAPP_OK;
        }
    }
    s = rollout_sub(c, kind, d_agents, d_agents_out, n_agents, goal, g, dt, steps, (cudaStream_t)stream);
    c->last_n_agents = n_agents;
    c->info.selection_fused = c->sel_fused ? 1 : 0;
    return s;
}

// one launch over n_agents agents (all of them, or the agents c->sub_idx lists)
static gmapp_status rollout_sub(gmapp_ctx* c, gmapp_kind kind, const float* d_agents, float* d_agents_out, int n_agents,
                                const float* goal, const gmapp_gains* g, float dt, int steps, cudaStream_t stream) {
    gmapp_status s;
    const int ng = kind == GMAPP_POINT3 ? 3 : 8;
    if (kind == GMAPP_POINT3 && !(c->has_tuning && c->tuning.scalar_path))
        return launch_rollout_x2(c, d_agents, d_agents_out, n_agents, goal, g, dt, steps, (cudaStream_t)stream);
    LaunchCfg cfg;
    s = choose_launch(c, kind, n_agents, &cfg);
    if (s != GMAPP_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    int launches = 0;
    RolloutParams P;
    memset(&P, 0, sizeof P);
    s = effective_spheres(c, g->r_agent, st, &P.sph, &launches);
    if (s != GMAPP_OK) return s;
    P.svel = c->d_svel;
    P.n_pad = cfg.n_pad;
    P.agents_in = d_agents; P.agents_out = d_agents_out;
    P.n_agents = n_agents; P.agents_per_cta = cfg.agents_per_cta;
    P.L = cfg.L; P.logL = ilog2(cfg.L);
    P.steps = steps;
    for (int i = 0; i < ng; ++i) P.goal[i] = goal[i];
    P.dt = dt; P.t0 = c->roll_t0;
    P.k_circ = g->k_circ; P.k_att = g->k_att; P.k_damp = g->k_damp;
    P.k_att_rot = g->k_att_rot; P.k_damp_rot = g->k_damp_rot;
    P.c_lin = g->vel_factor * dt * g->inv_mass;
    P.c_rot = g->vel_factor * dt * g->inv_inertia;
    P.inv_mass = g->inv_mass;
    P.r_d = g->r_influence; P.eps = g->eps_dist;
    P.apf = g->heuristic == 1;
    P.rcg = g->r_cost_goal > 0.0f ? g->r_cost_goal : g->r_influence;
    P.rco = g->r_cost_obs > 0.0f ? g->r_cost_obs : g->r_influence;
    P.rcg_is_rd = !(g->r_cost_goal > 0.0f); P.rco_is_rd = !(g->r_cost_obs > 0.0f);
    P.w_goal = g->w_goal; P.w_obs = g->w_obs; P.w_path = g->w_path; P.w_smooth = g->w_smooth;
    P.a_max = g->a_max; P.vel_factor = g->vel_factor;
    P.cost = c->d_cost; P.minclr = c->d_minclr; P.collided = c->d_collided;
    P.agent_idx = c->sub_idx;
    P.snap_out = c->roll_snap; P.snap_step = c->roll_snap_step; P.traj_out = c->roll_traj;
    P.count_dev = c->built_world ? c->d_vox_count : nullptr; P.n_cap = c->n_spheres;
    P.rd_arr = (c->ap_n > 0 && c->ap_has_rd) ? c->d_ap_rd : nullptr;
    P.kf_arr = (c->ap_n > 0 && c->ap_has_kf) ? c->d_ap_kf : nullptr;
    P.tile_off = cfg.tile_off; P.red_off = cfg.red_off;
    // few agents per CTA and many lanes per agent: sweep warps + one epilogue warp per group (gmapp_rollout_wide.cuh)
    const bool scalar_forced = c->has_tuning && c->tuning.scalar_path;
    const int n2 = (c->n_spheres + 1) / 2;
    bool wide = !scalar_forced && kind == GMAPP_MOTOR6 && cfg.groups <= 4 && cfg.L >= 64 && n2 >= 64;
    if (wide) {
        while (cfg.groups * cfg.L > 512 || cfg.L > pow2_ceil(n2)) cfg.L >>= 1;
        P.L = cfg.L; P.logL = ilog2(cfg.L);
        P.two_warp_epi = cfg.groups <= 3 ? 1 : 0;
        cfg.block = cfg.groups * cfg.L + (P.two_warp_epi ? 64 : 32) * cfg.groups;
        s = effective_pairs(c, g->r_agent, st, &launches);
        if (s != GMAPP_OK) return s;
        P.pairA = c->d_pairA; P.pair_stride = c->cap_spheres / 2; P.n2p = round_up(n2, cfg.L);
        // exchange area: per group the per-lane partials + the published states ((L + 8) float4), then one 5-float4
        // record per group for the ROT -> LIN hand-over
        cfg.tile_off = cfg.red_off + round_up((cfg.groups * (cfg.L + 8) + 5 * cfg.groups) * 16, 128);
        P.tile_off = cfg.tile_off;
        const size_t tile_bytes = (size_t)P.n2p * 16 * (c->moving ? 4 : 2);
        const bool fits = cfg.tile_off + tile_bytes <= (size_t)c->smem_optin;
        if (cfg.stage == 1 && !fits) cfg.stage = 0;
        cfg.smem = cfg.tile_off + (cfg.stage == 1 ? (int)tile_bytes : 0);
    }
    P.stage = cfg.stage;
    if (wide && c->sel_want && !c->sub_idx && GMAPP_FUSED_SELECT_WIDE) {             // the wide kernel has the fused selection tail, the scalar one does not
        P.sel.ticket = c->d_sel_ticket; P.sel.total = c->sel_total; P.sel.alpha = c->sel_alpha; P.sel.prev = c->sel_prev;
        P.sel.prev_dev = c->sel_prev_dev; P.sel.out_dev = c->d_sel_rec; P.sel.out_host = c->h_best; P.sel.seq = c->sel_seq;
        c->sel_fused = true;
    }
    rollout_fn fn = wide ? rollout_wide_kernel(c->moving, cfg.cull != 0, cfg.stage, g->heuristic == 1)
                         : rollout_kernel(kind, cfg.at, c->moving, cfg.cull != 0, cfg.stage);
    fn<<<cfg.grid, cfg.block, cfg.smem, st>>>(P);
    CUDA_TRY(c, cudaGetLastError());
    ++launches;
    c->last_n_agents = n_agents;
    gmapp_launch_info& I = c->info;
    I.grid = cfg.grid; I.block = cfg.block; I.lanes_per_agent = cfg.L; I.agents_per_thread = cfg.at;
    I.agents_per_cta = cfg.agents_per_cta; I.cull = cfg.cull; I.stage = cfg.stage;
    I.tile_spheres = cfg.stage == 1 ? cfg.n_pad : 0; I.n_tiles = cfg.stage == 1 ? 1 : 0;
    I.smem_bytes = cfg.smem; I.kernels_launched = launches; I.packed_x2 = 0;
    cudaFuncAttributes fa;
    if (cudaFuncGetAttributes(&fa, (const void*)fn) == cudaSuccess) I.regs_per_thread = fa.numRegs;
    return GMAPP_OK;
}

// ---------------------------------------------------------------------------------------------
// selection, force query, results
// ---------------------------------------------------------------------------------------------
// the selection record for (alpha, prev_best): from the rollout's fused tail when it was armed with the same
// arguments (or no incumbent is asked for: the raw argmin is in every record), else by the selection kernel
static gmapp_status selection_record_host(gmapp_ctx* c, float alpha, int prev_best, cudaStream_t st, const char* who) {
    if (c->last_n_agents < 1) return fail(c, GMAPP_ESTATE, "%s: no rollout has run on this context", who);
    if (!isfinite(alpha)) return fail(c, GMAPP_EINVAL, "%s: alpha is not finite", who);
    if (prev_best >= c->last_n_agents) prev_best = -1;        // not an agent of the last rollout: no incumbent
    const bool from_tail = c->sel_fused && !c->fused_prev_dev &&
                           (prev_best < 0 || (prev_best == c->fused_prev && alpha == c->fused_alpha));
    if (!from_tail) {
        // the kernel writes its record straight into pinned host memory (no copy engine round trip) and is launched
        // with programmatic stream serialisation, so its launch overlaps the tail of the rollout
        cudaLaunchConfig_t lc;
        memset(&lc, 0, sizeof lc);
        lc.gridDim = dim3(1); lc.blockDim = dim3(1024); lc.dynamicSmemBytes = 0; lc.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        lc.attrs = at; lc.numAttrs = 1;
        c->sel_seq = (c->sel_seq % 0x3fffffff) + 1;
        CUDA_TRY(c, cudaLaunchKernelEx(&lc, k_best_agent, (const float*)c->d_cost, (const int*)c->d_collided, c->last_n_agents, alpha,
                                       prev_best, (const int*)nullptr, c->d_sel_rec, c->h_best, c->sel_seq));
        c->sel_fused = false;                              // the record now belongs to this (alpha, prev_best)
    }
    {
        // The record is written to pinned memory by the rollout kernel's last warp (or by the selection kernel), the sequence number behind it: poll
        // for it instead of paying a stream synchronisation's wake-up latency.  Every few thousand polls look at the
        // stream: an error ends the wait, and a stream that has drained without the number appearing (it cannot) falls
        // through to the plain synchronise below.
        volatile int* flag = (volatile int*)(c->h_best + 8);
        for (unsigned spin = 1; *flag != c->sel_seq; ++spin) {
            if ((spin & 0x3fffu) == 0) {
                cudaError_t q = cudaStreamQuery(st);
                if (q != cudaErrorNotReady) {
                    if (q != cudaSuccess) return fail(c, GMAPP_ECUDA, "%s: the rollout failed", who);
                    break;
                }
            }
        }
        if (*flag != c->sel_seq) CUDA_TRY(c, cudaStreamSynchronize(st));
    }
    if (from_tail && prev_best < 0 && c->fused_prev >= 0) {    // armed with an incumbent, asked without: the raw argmin
        c->h_best[0] = c->h_best[3]; c->h_best[1] = c->h_best[4]; c->h_best[2] = c->h_best[5];
        c->fused_prev = -1;
    }
    return GMAPP_OK;
}

extern "C" gmapp_status gmapp_best_agent_ex(gmapp_ctx* c, float alpha, int prev_best, int* out_index, float* out_cost,
                                            int* out_collided, void* stream) {
    if (!c) return GMAPP_EINVAL;
    if (!out_index) return fail(c, GMAPP_EINVAL, "best_agent: out_index is NULL%s");
    gmapp_status s = selection_record_host(c, alpha, prev_best, (cudaStream_t)stream, "best_agent");
    if (s != GMAPP_OK) return s;
    *out_index = c->h_best[0];
    if (out_collided) *out_collided = c->h_best[1];
    if (out_cost) memcpy(out_cost, &c->h_best[2], sizeof(float));
    return GMAPP_OK;
}

extern "C" gmapp_status gmapp_select(gmapp_ctx* c, float alpha, int prev_best, gmapp_selection* out, void* stream) {
    if (!c) return GMAPP_EINVAL;
    if (!out) return fail(c, GMAPP_EINVAL, "select: out is NULL%s");
    gmapp_status s = selection_record_host(c, alpha, prev_best, (cudaStream_t)stream, "select");
    if (s != GMAPP_OK) return s;
    out->index = c->h_best[0]; out->collided = c->h_best[1]; memcpy(&out->cost, &c->h_best[2], sizeof(float));
    out->raw_index = c->h_best[3]; out->raw_collided = c->h_best[4]; memcpy(&out->raw_cost, &c->h_best[5], sizeof(float));
    out->prev_collided = c->h_best[6]; memcpy(&out->prev_cost, &c->h_best[7], sizeof(float));
    return GMAPP_OK;
}

extern "C" gmapp_status gmapp_set_selection(gmapp_ctx* c, float alpha, int prev_best) {
    if (!c) return GMAPP_EINVAL;
    if (!isfinite(alpha)) return fail(c, GMAPP_EINVAL, "set_selection: alpha is not finite%s");
    if (prev_best >= c->max_agents) return fail(c, GMAPP_EINVAL, "set_selection: prev_best exceeds max_agents%s");
    c->sel_alpha = alpha; c->sel_prev = prev_best < 0 ? -1 : prev_best;
    return GMAPP_OK;
}

extern "C" gmapp_status gmapp_best_agent(gmapp_ctx* c, float alpha, int prev_best, int* out_index, float* out_cost,
                                         void* stream) {
    return gmapp_best_agent_ex(c, alpha, prev_best, out_index, out_cost, nullptr, stream);
}

// ---------------------------------------------------------------------------------------------
// closed-loop re-planning (NEXT row N4): n_cycles planning cycles chained on the device
// ---------------------------------------------------------------------------------------------
extern "C" gmapp_status gmapp_set_trajectory_output(gmapp_ctx* c, float* d_traj) {
    if (!c) return GMAPP_EINVAL;
    c->roll_traj = d_traj;
    return GMAPP_OK;
}

extern "C" gmapp_status gmapp_replan(gmapp_ctx* c, gmapp_kind kind, float* d_agents, int n_agents, const float* goal,
                                     const gmapp_gains* g, float dt, int steps, int exec_steps, float alpha, int prev_best,
                                     int n_cycles, float* d_path_out, int32_t* d_best_out, void* stream) {
    if (!c) return GMAPP_EINVAL;
    if (!d_agents || !goal) return fail(c, GMAPP_EINVAL, "replan: NULL agents or goal%s");
    if (kind != GMAPP_POINT3 && kind != GMAPP_MOTOR6) return fail(c, GMAPP_EINVAL, "replan: unknown kind%s");
    if (n_cycles < 1) return fail(c, GMAPP_EINVAL, "replan: n_cycles must be >= 1%s");
    if (steps < 1 || exec_steps < 1 || exec_steps > steps) return fail(c, GMAPP_EINVAL, "replan: need 1 <= exec_steps <= steps%s");
    if (!isfinite(alpha)) return fail(c, GMAPP_EINVAL, "replan: alpha is not finite%s");
    if (n_agents < 1) return fail(c, GMAPP_EINVAL, "replan: n_agents must be >= 1%s");
    if (n_agents > c->max_agents) return fail(c, GMAPP_ECAPACITY, "replan: n_agents = %s%ld exceeds max_agents = %ld", "", n_agents, c->max_agents);
    if (prev_best >= n_agents) return fail(c, GMAPP_EINVAL, "replan: prev_best out of range%s");
    // everything gmapp_rollout would refuse is refused here, BEFORE the first enqueue (on error nothing is launched)
    if (!isfinite(dt) || !(dt > 0.0f)) return fail(c, GMAPP_EINVAL, "replan: dt must be finite and > 0%s");
    if (c->n_spheres < 0) return fail(c, GMAPP_ESTATE, "replan: gmapp_set_obstacles has not been called%s");
    gmapp_status s = check_gains(c, g, "replan");
    if (s != GMAPP_OK) return s;
    for (int i = 0; i < (kind == GMAPP_POINT3 ? 3 : 8); ++i) if (!isfinite(goal[i])) return fail(c, GMAPP_EINVAL, "replan: non-finite goal%s");
    if (c->ap_n > 0) {
        if (c->ap_n != n_agents) return fail(c, GMAPP_EINVAL, "replan: gmapp_set_agent_params was given %s%ld agents, the rollout %ld", "", c->ap_n, n_agents);
        if (c->ap_has_rd && g->eps_dist > c->ap_min_rd) return fail(c, GMAPP_EINVAL, "replan: need eps_dist <= every per-agent r_influence%s");
    }
    s = check_launchable(c, kind, n_agents);
    if (s != GMAPP_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    const int w = kind == GMAPP_POINT3 ? 6 : 14;
    // the incumbent goes to the device by a tiny kernel argument, not a host copy, so the whole call can be captured
    // in a CUDA graph and replayed
    k_set_int<<<1, 1, 0, st>>>(c->d_prev, prev_best < 0 ? -1 : prev_best);
    const float keep_alpha = c->sel_alpha; const int keep_prev = c->sel_prev;
    c->sel_alpha = alpha; c->sel_prev = -1; c->sel_prev_dev = c->d_prev;     // the rollouts' fused tails read the incumbent on the device
    int launches = 1;
    for (int cyc = 0; cyc < n_cycles && s == GMAPP_OK; ++cyc) {
        c->roll_t0 = (float)cyc * (float)exec_steps * dt;      // moving obstacles keep moving between cycles
        c->roll_snap = c->d_snap; c->roll_snap_step = exec_steps;
        s = gmapp_rollout(c, kind, d_agents, nullptr, n_agents, goal, g, dt, steps, stream);
        c->roll_t0 = 0.0f; c->roll_snap = nullptr; c->roll_snap_step = 0;
        if (s != GMAPP_OK) break;
        launches += c->info.kernels_launched;
        if (!c->sel_fused) {                                   // kernels without the fused tail (scalar path)
            k_best_agent<<<1, 1024, 0, st>>>(c->d_cost, c->d_collided, n_agents, alpha, -1, c->d_prev, c->d_sel_rec, nullptr, 0);
            ++launches;
        }
        k_reseed<<<(n_agents * w + 255) / 256, 256, 0, st>>>(c->d_snap, c->d_sel_rec, n_agents, w, d_agents, c->d_prev,
                                                             d_path_out, d_best_out, cyc);
        if (cudaGetLastError() != cudaSuccess) { s = fail(c, GMAPP_ECUDA, "replan: kernel launch failed%s"); break; }
        ++launches;
    }
    c->sel_alpha = keep_alpha; c->sel_prev = keep_prev; c->sel_prev_dev = nullptr;
    c->sel_fused = false;                                      // the record on the host side belongs to no (alpha, prev_best)
    c->info.kernels_launched = launches;
    return s;
}

extern "C" gmapp_status gmapp_forces(gmapp_ctx* c, gmapp_kind kind, const float* d_agents, int n_agents, const float* goal,
                                     const gmapp_gains* g, float t_obstacles, float* d_f_rep, float* d_f_total, void* stream) {
    if (!c) return GMAPP_EINVAL;
    if (kind != GMAPP_POINT3 && kind != GMAPP_MOTOR6) return fail(c, GMAPP_EINVAL, "forces: unknown kind%s");
    if (!d_agents || !goal) return fail(c, GMAPP_EINVAL, "forces: NULL agents or goal%s");
    if (n_agents < 1) return fail(c, GMAPP_EINVAL, "forces: n_agents must be >= 1%s");
    if (!isfinite(t_obstacles)) return fail(c, GMAPP_EINVAL, "forces: t_obstacles is not finite%s");
    if (c->n_spheres < 0) return fail(c, GMAPP_ESTATE, "forces: gmapp_set_obstacles has not been called%s");
    gmapp_status s = check_gains(c, g, "forces");
    if (s != GMAPP_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    ForceParams P;
    memset(&P, 0, sizeof P);
    s = effective_spheres(c, g->r_agent, st, &P.sph, nullptr);
    if (s != GMAPP_OK) return s;
    P.svel = c->d_svel;
    P.n_pad = c->n_spheres > 0 ? round_up(c->n_spheres, 32) : 0;
    P.agents = d_agents; P.n_agents = n_agents; P.kind = (int)kind;
    for (int i = 0; i < (kind == GMAPP_POINT3 ? 3 : 8); ++i) P.goal[i] = goal[i];
    P.k_circ = g->k_circ; P.k_att = g->k_att; P.k_damp = g->k_damp;
    P.k_att_rot = g->k_att_rot; P.k_damp_rot = g->k_damp_rot;
    P.r_d = g->r_influence; P.eps = g->eps_dist; P.t_obs = t_obstacles;
    P.apf = g->heuristic == 1; P.inv_rd = 1.0f / g->r_influence;
    P.f_rep = d_f_rep; P.f_total = d_f_total;
    const int warps_per_block = 8;
    const int grid = (n_agents + warps_per_block - 1) / warps_per_block;
    if (c->moving) k_forces<true><<<grid, 256, 0, st>>>(P);
    else k_forces<false><<<grid, 256, 0, st>>>(P);
    CUDA_TRY(c, cudaGetLastError());
    return GMAPP_OK;
}

extern "C" gmapp_status gmapp_get_results(gmapp_ctx* c, float* d_cost, float* d_min_clearance, int32_t* d_collided, void* stream) {
    if (!c) return GMAPP_EINVAL;
    if (c->last_n_agents < 1) return fail(c, GMAPP_ESTATE, "get_results: no rollout has run on this context%s");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = c->last_n_agents;
    if (d_cost) CUDA_TRY(c, cudaMemcpyAsync(d_cost, c->d_cost, sizeof(float) * 5 * n, cudaMemcpyDeviceToDevice, st));
    if (d_min_clearance) CUDA_TRY(c, cudaMemcpyAsync(d_min_clearance, c->d_minclr, sizeof(float) * n, cudaMemcpyDeviceToDevice, st));
    if (d_collided) CUDA_TRY(c, cudaMemcpyAsync(d_collided, c->d_collided, sizeof(int) * n, cudaMemcpyDeviceToDevice, st));
    return GMAPP_OK;
}

// ---------------------------------------------------------------------------------------------
// whole cycle from host buffers
// ---------------------------------------------------------------------------------------------
extern "C" gmapp_status gmapp_plan_cycle_host(gmapp_ctx* c, gmapp_kind kind, const float* h_agents, float* h_agents_out,
                                              int n_agents, const float* h_xyzr, const float* h_vel, int n_spheres,
                                              const float* goal, const gmapp_gains* g, float dt, int steps,
                                              float alpha, int prev_best, int* out_index, float* out_cost, void* stream) {
    if (!c) return GMAPP_EINVAL;
    if (!h_agents || !out_index || !goal) return fail(c, GMAPP_EINVAL, "plan_cycle_host: NULL agents, goal or out_index%s");
    if (kind != GMAPP_POINT3 && kind != GMAPP_MOTOR6) return fail(c, GMAPP_EINVAL, "plan_cycle_host: unknown kind%s");
    if (n_agents < 1 || steps < 1) return fail(c, GMAPP_EINVAL, "plan_cycle_host: n_agents and steps must be >= 1%s");
    if (n_agents > c->max_agents) return fail(c, GMAPP_ECAPACITY, "plan_cycle_host: n_agents = %s%ld exceeds max_agents = %ld", "", n_agents, c->max_agents);
    if (!isfinite(dt) || !(dt > 0.0f)) return fail(c, GMAPP_EINVAL, "plan_cycle_host: dt must be finite and > 0%s");
    if (!isfinite(alpha)) return fail(c, GMAPP_EINVAL, "plan_cycle_host: alpha is not finite%s");
    if (prev_best >= n_agents) return fail(c, GMAPP_EINVAL, "plan_cycle_host: prev_best out of range%s");
    if (n_spheres > 0 && !h_xyzr) return fail(c, GMAPP_EINVAL, "plan_cycle_host: n_spheres > 0 needs h_xyzr%s");
    if (n_spheres > c->max_spheres) return fail(c, GMAPP_ECAPACITY, "plan_cycle_host: n_spheres = %s%ld exceeds max_spheres = %ld", "", n_spheres, c->max_spheres);
    if (n_spheres < 0 && c->n_spheres < 0) return fail(c, GMAPP_ESTATE, "plan_cycle_host: no resident sphere world to keep (n_spheres < 0)%s");
    gmapp_status s = check_gains(c, g, "plan_cycle_host");
    if (s != GMAPP_OK) return s;
    // n_spheres < 0: keep the resident sphere world; n_spheres == 0: an EMPTY world (no obstacles); > 0: upload
    if (n_spheres >= 0) {
        s = gmapp_set_obstacles_host(c, h_xyzr, h_vel, n_spheres, stream);
        if (s != GMAPP_OK) return s;
    }
    const int w = kind == GMAPP_POINT3 ? 6 : 14;
    float* hp = c->h_pinned + (size_t)c->cap_spheres * 7;
    // every earlier use of the agent staging area ended with a stream synchronise (this call is synchronous)
    memcpy(hp, h_agents, sizeof(float) * w * (size_t)n_agents);
    // the rollout reads every start state once and writes every final state once: it does both straight from / to
    // the pinned host buffer (unified addressing), which saves two copy-engine transfers per cycle.  The selection is
    // armed with this call's (alpha, prev_best) and runs in the tail of the rollout kernel.
    const float keep_alpha = c->sel_alpha; const int keep_prev = c->sel_prev;
    c->sel_alpha = alpha; c->sel_prev = prev_best < 0 ? -1 : prev_best;
    s = gmapp_rollout(c, kind, hp, h_agents_out ? hp : nullptr, n_agents, goal, g, dt, steps, stream);
    c->sel_alpha = keep_alpha; c->sel_prev = keep_prev;
    if (s != GMAPP_OK) return s;
    s = gmapp_best_agent(c, alpha, prev_best, out_index, out_cost, stream);     // synchronises
    if (s != GMAPP_OK) return s;
    if (h_agents_out) memcpy(h_agents_out, hp, sizeof(float) * w * (size_t)n_agents);
    return GMAPP_OK;
}

// ---------------------------------------------------------------------------------------------
// FP32 peak microbenchmark
// ---------------------------------------------------------------------------------------------
extern "C" gmapp_status gmapp_measure_fp32_peak(gmapp_ctx* c, int use_f32x2, float* out_tflops, void* stream) {
    if (!c || !out_tflops) return GMAPP_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int grid = c->num_sms * 8, block = 256, iters = 2048;
    float best_ms = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        CUDA_TRY(c, cudaEventRecord(c->ev0, st));
        if (use_f32x2) k_fma_peak<true><<<grid, block, 0, st>>>(c->d_scratch, iters, 1.0000001f, 1e-9f);
        else k_fma_peak<false><<<grid, block, 0, st>>>(c->d_scratch, iters, 1.0000001f, 1e-9f);
        CUDA_TRY(c, cudaGetLastError());
        CUDA_TRY(c, cudaEventRecord(c->ev1, st));
        CUDA_TRY(c, cudaEventSynchronize(c->ev1));
        float ms = 0.0f;
        CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev0, c->ev1));
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    const double fmas = (double)grid * block * (double)iters * 128.0;
    *out_tflops = (float)(2.0 * fmas / (best_ms * 1e-3) / 1e12);
    return GMAPP_OK;
}

// ---------------------------------------------------------------------------------------------
// issue-cost microbenchmarks (gmapp_microbench.cuh)
// ---------------------------------------------------------------------------------------------
extern "C" gmapp_status gmapp_microbench(gmapp_ctx* c, int kind, float* out_cycles, void* stream) {
    if (!c || !out_cycles) return GMAPP_EINVAL;
    if (kind < 0 || kind >= MB_COUNT) return fail(c, GMAPP_EINVAL, "microbench: kind must be 0..%s%ld", "", (long)MB_COUNT - 1);
    cudaStream_t st = (cudaStream_t)stream;
    int clock_khz = 0;
    CUDA_TRY(c, cudaDeviceGetAttribute(&clock_khz, cudaDevAttrClockRate, c->device));
    const int iters = 20000;
    float best_ms = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        CUDA_TRY(c, cudaEventRecord(c->ev0, st));
        const float a = 0.999f, b = 1e-3f, thr = 1e30f;
        switch (kind) {
#define MB_CASE(K) case K: k_microbench<K><<<c->num_sms, 512, 0, st>>>(c->d_scratch, iters, a, b, thr); break;
            MB_CASE(0) MB_CASE(1) MB_CASE(2) MB_CASE(3) MB_CASE(4) MB_CASE(5) MB_CASE(6) MB_CASE(7) MB_CASE(8) MB_CASE(9) MB_CASE(10) MB_CASE(11) MB_CASE(12) MB_CASE(13) MB_CASE(14)
#undef MB_CASE
        }
        CUDA_TRY(c, cudaGetLastError());
        CUDA_TRY(c, cudaEventRecord(c->ev1, st));
        CUDA_TRY(c, cudaEventSynchronize(c->ev1));
        float ms = 0.0f;
        CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev0, c->ev1));
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    // cycles per warp-instruction per SM sub-partition at the device's maximum SM clock: 4 warps x iters x 8 instructions
    *out_cycles = (float)((double)best_ms * 1e-3 * (double)clock_khz * 1e3 / (4.0 * iters * 8.0));
    return GMAPP_OK;
}

// ---------------------------------------------------------------------------------------------
// Allocation-free entry point: the sphere-world builder with its scratch in a file-scope static device array.
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
// no context, no cudaMalloc / cudaFree / allocating library routine anywhere on this path.
//
// The scratch -- the voxel bitmap of the largest grid this entry point accepts, kStaticMaxVoxels = 262 144 voxels = 8192
// words, plus the finished-block counter -- is g_static_scratch below: 33 024 bytes that EVERY GPU that loads the library
// holds until the process exits.  In host code the array's NAME is a host-side stand-in, not a device address: the
// address is fetched once per device, with that device current, by cudaGetSymbolAddress, and that pointer is what the
// kernel gets.  All calls (of every thread, on every stream) share the one array of a device: it is cleared at the start
// of every call (stream-ordered memset; it also keeps the previous call's contents otherwise), and two calls whose
// stream work OVERLAPS on the same GPU race on it -- keep calls on one stream, or order them yourself.
// ---------------------------------------------------------------------------------------------
constexpr int kStaticMaxVoxels = kVoxSmallWords * 32;
constexpr int kStaticScratchWords = kVoxSmallWords + 64;     // bitmap words, then the counter (padded to 256 bytes)
static __device__ __align__(256) unsigned g_static_scratch[kStaticScratchWords];

// the small-grid build of gmapp_voxel.cuh writing only a caller-owned (x, y, z, r) array: per-block bitmaps in shared
// memory, merged into the scratch bitmap; the block that finishes last scans it and emits the spheres over the sentinels
__global__ void __launch_bounds__(1024) k_vox_build_static(const float* __restrict__ pts, int n_points, const __grid_constant__ VoxelGrid G,
                                                           unsigned* scratch, int capacity, float4* xyzr_out, int* count_out) {
    extern __shared__ unsigned sbits[];                      // [n_words] this block's bitmap; the last block: the merged one
    __shared__ int s[32];
    __shared__ int s_last;
    unsigned* bitmap = scratch;
    int* done = reinterpret_cast<int*>(scratch + kVoxSmallWords);
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5, nw = G.n_words;
    for (int w = t; w < nw; w += 1024) sbits[w] = 0u;
    __syncthreads();
    for (int i = blockIdx.x * 1024 + t; i < n_points; i += gridDim.x * 1024) {
        const int v = vox_of_point(pts, i, G);
        if (v >= 0) {
            const unsigned bit = 1u << (v & 31);
            if (!(sbits[v >> 5] & bit)) atomicOr(&sbits[v >> 5], bit);
        }
    }
    for (int i = blockIdx.x * 1024 + t; i < capacity; i += gridDim.x * 1024) xyzr_out[i] = make_float4(kFar, kFar, kFar, 0.0f);
    __syncthreads();
    for (int w = t; w < nw; w += 1024) {
        const unsigned m = sbits[w];
        if (m && (m & ~__ldcg(&bitmap[w]))) atomicOr(&bitmap[w], m);
    }
    __threadfence();
    __syncthreads();
    if (t == 0) s_last = (atomicAdd(done, 1) == int(gridDim.x) - 1) ? 1 : 0;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int per = (nw + 1023) / 1024;                      // thread t owns the contiguous words [t per, t per + per)
    int mine = 0;
    for (int k = 0; k < per; ++k) {
        const int w = t * per + k;
        if (w < nw) { const unsigned m = __ldcg(&bitmap[w]); sbits[w] = m; mine += __popc(m); }
    }
    int inc = mine;
    for (int off = 1; off < 32; off <<= 1) { int o = __shfl_up_sync(0xffffffffu, inc, off); if (lane >= off) inc += o; }
    if (lane == 31) s[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int ws = s[lane], wi = ws;
        for (int off = 1; off < 32; off <<= 1) { int o = __shfl_up_sync(0xffffffffu, wi, off); if (lane >= off) wi += o; }
        s[lane] = wi - ws;
        if (lane == 31 && count_out) *count_out = wi;
    }
    __syncthreads();
    int rank = s[wid] + inc - mine;
    for (int k = 0; k < per; ++k) {
        const int w = t * per + k;
        if (w >= nw) break;
        unsigned bits = sbits[w];
        while (bits) {
            const int bpos = __ffs(bits) - 1;
            bits &= bits - 1;
            if (rank < capacity) xyzr_out[rank] = vox_sphere((unsigned(w) << 5) + bpos, G);
            ++rank;
        }
    }
}

#include <mutex>
namespace {
struct StaticDev { bool ready; unsigned* scratch; int sms; };
StaticDev g_static_dev[64];                                  // zero-initialised: not ready
std::mutex g_static_mutex;
}  // namespace

// once per device, with that device current: the DEVICE address of g_static_scratch and the SM count
static gmapp_status static_setup(int device, StaticDev* out) {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDev& d = g_static_dev[device];
    if (!d.ready) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) return fail(nullptr, GMAPP_ECUDA, "build_sphere_world_static: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e));
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
        if (e != cudaSuccess || sms < 1) return fail(nullptr, GMAPP_ECUDA, "build_sphere_world_static: cudaDeviceGetAttribute failed: %s", cudaGetErrorString(e));
        d.scratch = (unsigned*)p; d.sms = sms; d.ready = true;
    }
    *out = d;
    return GMAPP_OK;
}

extern "C" gmapp_status gmapp_build_sphere_world_static(int device, const float* d_points, int n_points, const float* lo,
                                                        const float* hi, float pitch, int capacity, float* d_xyzr_out,
                                                        int32_t* d_count_out, void* stream) {
    if (device < 0 || device >= 64) return fail(nullptr, GMAPP_EINVAL, "build_sphere_world_static: device must be 0..63%s");
    if (n_points < 0 || (n_points > 0 && !d_points) || !lo || !hi || !d_xyzr_out)
        return fail(nullptr, GMAPP_EINVAL, "build_sphere_world_static: NULL points / bounds / output or n_points < 0%s");
    if (((uintptr_t)d_xyzr_out & 15u) != 0) return fail(nullptr, GMAPP_EINVAL, "build_sphere_world_static: d_xyzr_out must be 16-byte aligned%s");
    if (!isfinite(pitch) || !(pitch > 0.0f)) return fail(nullptr, GMAPP_EINVAL, "build_sphere_world_static: pitch must be finite and > 0%s");
    if (capacity < 1 || capacity > (1 << 24)) return fail(nullptr, GMAPP_EINVAL, "build_sphere_world_static: capacity must be 1..2^24%s");
    VoxelGrid G;
    double nvox = 1.0;
    for (int a = 0; a < 3; ++a) {
        if (!isfinite(lo[a]) || !isfinite(hi[a]) || !(hi[a] > lo[a])) return fail(nullptr, GMAPP_EINVAL, "build_sphere_world_static: need finite lo < hi%s");
        G.lo[a] = lo[a]; G.hi[a] = hi[a];
        const double d = ceil(((double)hi[a] - (double)lo[a]) / (double)pitch);
        if (d > 4096.0) return fail(nullptr, GMAPP_ECAPACITY, "build_sphere_world_static: more than 4096 voxels along an axis (static scratch: %s%ld voxels in all)", "", (long)kStaticMaxVoxels);
        G.dim[a] = d < 1.0 ? 1 : (int)d;
        nvox *= G.dim[a];
    }
    if (nvox > (double)kStaticMaxVoxels)
        return fail(nullptr, GMAPP_ECAPACITY, "build_sphere_world_static: the voxel grid (%s%ld voxels) exceeds the static scratch of %ld voxels; "
                    "use gmapp_build_sphere_world", "", (long)nvox, (long)kStaticMaxVoxels);
    G.pitch = pitch;
    G.n_words = ((int)nvox + 31) / 32;
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return fail(nullptr, GMAPP_ECUDA, "build_sphere_world_static: cudaSetDevice: %s", cudaGetErrorString(e));
    StaticDev dev;
    gmapp_status s = static_setup(device, &dev);
    if (s != GMAPP_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    // the array keeps the last call's contents: the bitmap words and the counter must start at zero
    e = cudaMemsetAsync(dev.scratch, 0, sizeof(unsigned) * kStaticScratchWords, st);
    if (e != cudaSuccess) return fail(nullptr, GMAPP_ECUDA, "build_sphere_world_static: cudaMemsetAsync: %s", cudaGetErrorString(e));
    int grid = (n_points + 2047) / 2048;                    // two points per thread
    if (grid < 1) grid = 1;
    if (grid > 2 * dev.sms) grid = 2 * dev.sms;
    k_vox_build_static<<<grid, 1024, sizeof(unsigned) * G.n_words, st>>>(d_points, n_points, G, dev.scratch, capacity,
                                                                        reinterpret_cast<float4*>(d_xyzr_out), d_count_out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(nullptr, GMAPP_ECUDA, "build_sphere_world_static: kernel launch: %s", cudaGetErrorString(e));
    return GMAPP_OK;
}
