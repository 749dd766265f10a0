// gmapp_kernels.cuh -- the rollout / force / selection kernels (sm_100a, FP32).
//
// Thread mapping.  A "group" is L = lanes_per_agent consecutive threads (L a power of two).  A group
// owns AT (1 or 2) agents and keeps their state in registers for the whole rollout; lane l of the group
// evaluates spheres l, l+L, l+2L, ... at every step, so the sphere sum of an agent is split over the L
// lanes and combined once per step by a fixed-order xor-shuffle tree (plus a shared-memory exchange and
// one named barrier when the group spans several warps).  Every lane then integrates the group's
// agents redundantly, so no state is ever broadcast back; the group's first warp alone accumulates the
// costs.  Groups never wait for each other, so one group's reduce / integrate tail overlaps the other
// groups' pair loops on the same SM.  Reductions use no atomics and a fixed order: results are
// bit-reproducible run to run.
//
// Sphere staging.  STAGE 1: the whole packed sphere set (16 B per static sphere, +16 B velocity) is
// copied once per rollout into shared memory by 1-D TMA bulk copies completing on an mbarrier, and
// reused by every agent of the CTA for every step.  STAGE 0: spheres are read from global memory
// through L1/L2 (sets that exceed shared memory; round-1 fallback for the tile ring).
//
// Pair math (static spheres), per agent-sphere pair, branch-free:
//   d = c - p; q = |d|^2 (+1e-30 so q > 0); y = MUFU.RSQ(q); t = q y; dist = t + (y/2)(q - t^2)  (1 Newton step)
//   ds = dist - R (R = r_j + r_a packed at set-up); dmin = min(dmin, ds); dO = max(ds, eps)
//   s = d.v; w = s * MUFU.RCP(dO q); if (ds <= r_d) B += w d
// and once per agent-step  f_r = k_f [ ((B.v)/|v|) v - |v| B ]   (BAC-CAB form of Eq. 2-3).
// Moving spheres use the per-pair relative velocity and accumulate the force vector directly.
#pragma once
#include "gmapp_device.cuh"

namespace gmapp {

constexpr float kTiny = 1e-30f;          // bias that keeps squared norms > 0 (absorbed exactly otherwise)
// Sentinel spheres (padding of the sphere arrays) sit at (kFar, kFar, kFar) with radius 0: never gated, never the
// minimum, and far enough that every quantity derived from them stays FINITE in FP32 (|d|^2 ~ 3e12, d_O |d|^2 ~ 5e18).
// The sphere world and the agents must stay within |coordinate| <= 1e5 m of the origin.
constexpr float kFar = 1.0e6f;
constexpr int kMaxGroupsNamedBar = 15;   // named barriers 1..15

// Selection fused into the rollout's tail (S8, reading G24).  Every warp that has written the results of
// its agents takes a ticket; the warp that completes the count reduces (collided, C, index) over all agents, applies the
// hysteresis rule and writes the 8-word selection record -- no second launch in the planning cycle.
//   record: {index, collided, cost | raw index, raw collided, raw cost (plain argmin, no incumbent) | incumbent collided, cost}
struct SelParams {
    int* ticket;              // device counter (0 between cycles); nullptr: selection not fused into this launch
    int total;                // agents of the whole cycle (all launches of a heterogeneous ensemble together)
    float alpha;
    int prev;                 // incumbent, or < 0
    const int* prev_dev;      // nullable: the incumbent lives on the device (gmapp_replan)
    int* out_dev;             // [8] the record in device memory
    int* out_host;            // nullable: [9] the same record in pinned host memory, then `seq` (the host polls for it)
    int seq;                  // sequence number of this cycle
};

struct RolloutParams {
    const float4* sph;        // [n_pad] (cx, cy, cz, r_j + r_a), sentinel-padded
    const float4* svel;       // [n_pad] (ux, uy, uz, 0) or nullptr
    int n_pad;                // multiple of L
    const float4* pairA;      // sphere-pair arrays A, B, U, V (gmapp_rollout_wide.cuh), pair_stride float4 apart
    int pair_stride, n2p;     // n2p = sphere pairs padded to a multiple of L
    const float* agents_in;   // [n][6] or [n][14]
    float* agents_out;        // same layout or nullptr
    int n_agents, agents_per_cta;
    int L, logL;
    int steps;
    float goal[8];
    float dt;
    float k_circ, k_att, k_damp, k_att_rot, k_damp_rot;
    float c_lin, c_rot;       // vel_factor * dt * inv_mass, vel_factor * dt * inv_inertia  (Eq. 9-10)
    float inv_mass;
    float r_d, eps;
    float rcg, rco;           // Eq. 17 / 18 radii
    float w_goal, w_obs, w_path, w_smooth, a_max, vel_factor;
    float* cost;              // [n][5]
    float* minclr;            // [n]
    int* collided;            // [n]
    int apf;                  // 1: APF heuristic (Eq. 1) instead of the circular field (Eq. 2-3)
    // heterogeneous ensemble (gmapp_set_agent_params): all nullable
    const int* agent_idx;     // [n_agents] this launch's agents as indices into the caller's arrays
    const float* rd_arr;      // per-agent detection radius r_d, indexed by the caller's agent index
    const float* kf_arr;      // per-agent gain k_f
    int rcg_is_rd, rco_is_rd; // Eq. 17 / 18 radii default to the agent's own r_d
    int stage;                // gmapp_rollout_wide.cuh: 1 = pair arrays staged in shared memory (run-time choice)
    // closed-loop re-planning (gmapp_replan): obstacle time at step 0, and an optional state snapshot
    float t0;                 // obstacles are evaluated at t0 + k dt
    float* snap_out;          // [n][6|14] states after snap_step steps (indexed like agents_in), or nullptr
    int snap_step;            // 1..steps
    float* traj_out;          // nullable: [n][steps+1][6|14] every pose of every agent (pose 0 = start state, written by the host side)
    const int* count_dev;     // nullable: device-resident sphere count of a built sphere world (wide kernel only)
    int n_cap;
    int two_warp_epi;         // wide kernel, 6D agents: a rot warp and a lin warp per group (G <= 3)
    int tile_off;             // byte offset of the sphere tile in dynamic shared memory
    int red_off;              // byte offset of the cross-warp exchange scratch
    SelParams sel;            // selection fused into the tail (wide kernel only)
};

__device__ __forceinline__ int agent_gid(const RolloutParams& P, int i) { return P.agent_idx ? P.agent_idx[i] : i; }
__device__ __forceinline__ float agent_rd(const RolloutParams& P, int gid) { return P.rd_arr ? P.rd_arr[gid] : P.r_d; }
__device__ __forceinline__ float agent_kf(const RolloutParams& P, int gid) { return P.kf_arr ? P.kf_arr[gid] : P.k_circ; }

// ---------------------------------------------------------------------------------------------
// per-pair math
// ---------------------------------------------------------------------------------------------
template <int NA>
struct StaticAcc {            // per-lane partial sums for NA agents, static spheres
    float bx[NA], by[NA], bz[NA], dmin[NA];
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int a = 0; a < NA; ++a) { bx[a] = by[a] = bz[a] = 0.0f; dmin[a] = __int_as_float(0x7f800000); }
    }
};

// distance part shared by all variants: returns ds, leaves d, q
__device__ __forceinline__ float pair_distance(float cx, float cy, float cz, float R,
                                               float px, float py, float pz,
                                               float& dx, float& dy, float& dz, float& q) {
    dx = cx - px; dy = cy - py; dz = cz - pz;
    q = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, kTiny)));
    float y = rsqrt_approx(q);
    float t = q * y;
    float e = fmaf(-t, t, q);
    return fmaf(0.5f * y, e, t - R);
}

// APF (Eq. 1, Khatib form on the clamped surface distance, reading N1):
// f_j = -k_f (1/d_O - 1/r_d) / d_O^2 * d/|d|; accumulated without k_f; exactly 0 outside r_d
__device__ __forceinline__ void apf_accumulate(float ds, float q, float dx, float dy, float dz, float r_d, float eps,
                                               float& bx, float& by, float& bz) {
    if (ds <= r_d) {
        const float ro = rcp_approx(fmaxf(ds, eps));
        const float m = (rcp_approx(r_d) - ro) * (ro * ro) * rsqrt_approx(q);
        bx = fmaf(m, dx, bx); by = fmaf(m, dy, by); bz = fmaf(m, dz, bz);
    }
}

template <int NA, bool FORCE, bool CULL, bool APF = false>
__device__ __forceinline__ void pair_static(const float4 s, const float (&p)[NA][3], const float (&v)[NA][3],
                                            const float (&rd)[NA], float eps, unsigned mask, StaticAcc<NA>& acc) {
    float dx[NA], dy[NA], dz[NA], q[NA], ds[NA];
    bool any = false;
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        ds[a] = pair_distance(s.x, s.y, s.z, s.w, p[a][0], p[a][1], p[a][2], dx[a], dy[a], dz[a], q[a]);
        acc.dmin[a] = fminf(acc.dmin[a], ds[a]);
        any = any || (ds[a] <= rd[a]);
    }
    if (!FORCE) return;
    if (CULL) { if (!__any_sync(mask, any)) return; }
    if (APF) {
#pragma unroll
        for (int a = 0; a < NA; ++a) apf_accumulate(ds[a], q[a], dx[a], dy[a], dz[a], rd[a], eps, acc.bx[a], acc.by[a], acc.bz[a]);
        return;
    }
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        float dO = fmaxf(ds[a], eps);
        float sv = fmaf(dx[a], v[a][0], fmaf(dy[a], v[a][1], dz[a] * v[a][2]));
        float w = sv * rcp_approx(dO * q[a]);
        if (ds[a] <= rd[a]) {
            acc.bx[a] = fmaf(w, dx[a], acc.bx[a]);
            acc.by[a] = fmaf(w, dy[a], acc.by[a]);
            acc.bz[a] = fmaf(w, dz[a], acc.bz[a]);
        }
    }
}

// moving spheres: centre advected to obstacle time tk, relative velocity per pair, force accumulated
// directly:  f_j = w [ (s/|vr|) vr - |vr| d ],  w = s / (dO q),  s = d.vr   (k_f applied after the sum)
template <int NA, bool FORCE, bool CULL, bool APF = false>
__device__ __forceinline__ void pair_moving(const float4 s, const float4 su, float tk,
                                            const float (&p)[NA][3], const float (&v)[NA][3],
                                            const float (&rd)[NA], float eps, unsigned mask, StaticAcc<NA>& acc) {
    const float cx = fmaf(tk, su.x, s.x), cy = fmaf(tk, su.y, s.y), cz = fmaf(tk, su.z, s.z);
    float dx[NA], dy[NA], dz[NA], q[NA], ds[NA];
    bool any = false;
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        ds[a] = pair_distance(cx, cy, cz, s.w, p[a][0], p[a][1], p[a][2], dx[a], dy[a], dz[a], q[a]);
        acc.dmin[a] = fminf(acc.dmin[a], ds[a]);
        any = any || (ds[a] <= rd[a]);
    }
    if (!FORCE) return;
    if (CULL) { if (!__any_sync(mask, any)) return; }
    if (APF) {
#pragma unroll
        for (int a = 0; a < NA; ++a) apf_accumulate(ds[a], q[a], dx[a], dy[a], dz[a], rd[a], eps, acc.bx[a], acc.by[a], acc.bz[a]);
        return;
    }
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        float vx = v[a][0] - su.x, vy = v[a][1] - su.y, vz = v[a][2] - su.z;
        float n2 = fmaf(vx, vx, fmaf(vy, vy, fmaf(vz, vz, kTiny)));
        float inv = rsqrt_approx(n2);
        float nv = n2 * inv;
        float dO = fmaxf(ds[a], eps);
        float sv = fmaf(dx[a], vx, fmaf(dy[a], vy, dz[a] * vz));
        float w = sv * rcp_approx(dO * q[a]);
        float c1 = w * sv * inv, c2 = -w * nv;
        if (ds[a] <= rd[a]) {
            acc.bx[a] = fmaf(c1, vx, fmaf(c2, dx[a], acc.bx[a]));
            acc.by[a] = fmaf(c1, vy, fmaf(c2, dy[a], acc.by[a]));
            acc.bz[a] = fmaf(c1, vz, fmaf(c2, dz[a], acc.bz[a]));
        }
    }
}

// One lane's slice of the sphere sum for NA agents at obstacle time tk.
template <int NA, bool MOVING, bool FORCE, bool CULL, bool APF = false>
__device__ __forceinline__ void sphere_sweep(const float4* __restrict__ sph, const float4* __restrict__ svel,
                                             int n_pad, int lane, int L, float tk,
                                             const float (&p)[NA][3], const float (&v)[NA][3],
                                             const float (&rd)[NA], float eps, unsigned mask, StaticAcc<NA>& acc) {
    constexpr int U = (NA == 1) ? 4 : 2;
    int j = lane;
    const int step = L * U;
    for (; j + step - L < n_pad; j += step) {
        float4 s[U], su[U];
#pragma unroll
        for (int u = 0; u < U; ++u) { s[u] = sph[j + u * L]; if (MOVING) su[u] = svel[j + u * L]; }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (MOVING) pair_moving<NA, FORCE, CULL, APF>(s[u], su[u], tk, p, v, rd, eps, mask, acc);
            else        pair_static<NA, FORCE, CULL, APF>(s[u], p, v, rd, eps, mask, acc);
        }
    }
    for (; j < n_pad; j += L) {
        float4 s = sph[j];
        if (MOVING) pair_moving<NA, FORCE, CULL, APF>(s, svel[j], tk, p, v, rd, eps, mask, acc);
        else        pair_static<NA, FORCE, CULL, APF>(s, p, v, rd, eps, mask, acc);
    }
}

// ---------------------------------------------------------------------------------------------
// group all-reduce: sum of (bx,by,bz), min of dmin over the L lanes of a group; every lane gets the
// result.  Fixed order -> deterministic; fp add is commutative so xor partners agree bitwise.
// ---------------------------------------------------------------------------------------------
template <int NA>
__device__ __forceinline__ void group_allreduce(StaticAcc<NA>& acc, int L, int lane_in_group, int group_in_cta,
                                                float* red, int parity, unsigned mask) {
    const int wl = L < 32 ? L : 32;
    for (int off = wl >> 1; off > 0; off >>= 1) {
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            acc.bx[a] += __shfl_xor_sync(mask, acc.bx[a], off);
            acc.by[a] += __shfl_xor_sync(mask, acc.by[a], off);
            acc.bz[a] += __shfl_xor_sync(mask, acc.bz[a], off);
            acc.dmin[a] = fminf(acc.dmin[a], __shfl_xor_sync(mask, acc.dmin[a], off));
        }
    }
    if (L > 32) {
        // cross-warp exchange: red[parity][warp_in_cta][2 agents] float4; the group's warps are contiguous.
        // Double-buffered by step parity so one named barrier per step is enough (a warp can run at most
        // one barrier ahead of the slowest warp of its group).
        const int W = L >> 5;
        const int w0 = (group_in_cta * L) >> 5;
        float4* base = reinterpret_cast<float4*>(red) + (parity * 32 + w0) * 2;
        if ((lane_in_group & 31) == 0) {
            const int wig = lane_in_group >> 5;
#pragma unroll
            for (int a = 0; a < NA; ++a)
                base[wig * 2 + a] = make_float4(acc.bx[a], acc.by[a], acc.bz[a], acc.dmin[a]);
        }
        named_bar_sync(1 + group_in_cta, L);
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            float4 t = base[a];
            for (int w = 1; w < W; ++w) {
                float4 o = base[w * 2 + a];
                t.x += o.x; t.y += o.y; t.z += o.z; t.w = fminf(t.w, o.w);
            }
            acc.bx[a] = t.x; acc.by[a] = t.y; acc.bz[a] = t.z; acc.dmin[a] = t.w;
        }
    }
}

// circular-field force from the reduced sums (static spheres): f_r = k_f [ ((B.v)/|v|) v - |v| B ]
__device__ __forceinline__ void cf_force_static(float k_circ, float bx, float by, float bz,
                                                float vx, float vy, float vz, float& fx, float& fy, float& fz) {
    float n2 = fmaf(vx, vx, fmaf(vy, vy, fmaf(vz, vz, kTiny)));
    float inv = rsqrt_approx(n2);
    inv = inv * fmaf(-0.5f * n2 * inv, inv, 1.5f);        // Newton step: 1/|v| to ~1 ulp
    float nv = n2 * inv;
    float A = fmaf(bx, vx, fmaf(by, vy, bz * vz));
    float c1 = k_circ * A * inv, c2 = -k_circ * nv;
    fx = fmaf(c1, vx, c2 * bx); fy = fmaf(c1, vy, c2 * by); fz = fmaf(c1, vz, c2 * bz);
}

// ---------------------------------------------------------------------------------------------
// cost accumulators (Eq. 16-20), kept by the first warp of a group
// ---------------------------------------------------------------------------------------------
// Kahan-compensated add: the sums run over up to thousands of poses and must stay within 1e-5 absolute
__device__ __forceinline__ void kahan_add(float& s, float& c, float x) {
    float y = x - c;
    float t = s + y;
    c = (t - s) - y;
    s = t;
}

struct CostAcc {
    float sumG, cG, sumO, cO, sumV, cV, sumJ, cJ, minclr, d1;
    int collided;
    __device__ __forceinline__ void init(float dg) {
        sumG = cG = sumO = cO = sumV = cV = sumJ = cJ = 0.0f;
        minclr = __int_as_float(0x7f800000); d1 = dg; collided = 0;
    }
    // one pose: Eq. 17 / 18 summands (exactly 1 / exactly 0 when saturated), clearance and collision record
    __device__ __forceinline__ void pose(float dg, float dmin, float rcg, float rco) {
        kahan_add(sumG, cG, dg >= rcg ? 1.0f : dg / rcg);
        kahan_add(sumO, cO, dmin >= rco ? 0.0f : 1.0f - fmaxf(dmin, 0.0f) / rco);
        minclr = fminf(minclr, dmin);
        collided |= (dmin < 0.0f) ? 1 : 0;
    }
    __device__ __forceinline__ void add_len(float x) { kahan_add(sumV, cV, x); }
    __device__ __forceinline__ void add_jerk(float x) { kahan_add(sumJ, cJ, x); }
    __device__ __forceinline__ void finish(const RolloutParams& P, float L_path, float J, float* out5) const {
        const float Nk = float(P.steps) + 1.0f;
        float Cg = sumG / Nk;
        float Co = sumO / Nk;
        float Cp;
        if (L_path == 0.0f && d1 == 0.0f) Cp = 0.0f;
        else if (L_path >= d1) Cp = 1.0f - d1 / L_path;
        else Cp = 1.0f - L_path / d1;
        float dt2 = P.dt * P.dt;
        float Cs = fminf(1.0f, J / (Nk * dt2 * dt2 * P.a_max * P.a_max));
        out5[0] = P.w_goal * Cg + P.w_obs * Co + P.w_path * Cp + P.w_smooth * Cs;
        out5[1] = Cg; out5[2] = Co; out5[3] = Cp; out5[4] = Cs;
    }
};

__device__ __forceinline__ float norm3f(float x, float y, float z) {
    float n2 = fmaf(x, x, fmaf(y, y, fmaf(z, z, kTiny)));
    float inv;
    float n = sqrt_refined(n2, inv);
    return n2 <= kTiny ? 0.0f : n;
}

// ---------------------------------------------------------------------------------------------
// 3D point agents
// ---------------------------------------------------------------------------------------------
template <int NA, bool MOVING, bool CULL>
__device__ __forceinline__ void rollout_point3(const RolloutParams& P, const float4* sph, const float4* svel,
                                               int first_agent, int lane_in_group, int group_in_cta, float* red) {
    const unsigned mask = __activemask();      // lanes of this warp on this code path (sub-warp groups may differ)
    float p[NA][3], v[NA][3], rd[NA], kf[NA];
    int gid[NA];
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        gid[a] = agent_gid(P, first_agent + a); rd[a] = agent_rd(P, gid[a]); kf[a] = agent_kf(P, gid[a]);
        const float* s = P.agents_in + 6 * size_t(gid[a]);
#pragma unroll
        for (int i = 0; i < 3; ++i) { p[a][i] = s[i]; v[a][i] = s[3 + i]; }
    }
    const bool cost_warp = lane_in_group < 32;
    CostAcc ca[NA];
    float ap[NA][3];                                      // previous acceleration (Eq. 20 via differences of a)
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        ca[a].init(norm3f(P.goal[0] - p[a][0], P.goal[1] - p[a][1], P.goal[2] - p[a][2]));
        ap[a][0] = ap[a][1] = ap[a][2] = 0.0f;
    }
    StaticAcc<NA> acc;
    for (int k = 0; k < P.steps; ++k) {
        const float tk = fmaf(float(k), P.dt, P.t0);
        acc.clear();
        if (P.apf) sphere_sweep<NA, MOVING, true, CULL, true>(sph, svel, P.n_pad, lane_in_group, P.L, tk, p, v, rd, P.eps, mask, acc);
        else sphere_sweep<NA, MOVING, true, CULL>(sph, svel, P.n_pad, lane_in_group, P.L, tk, p, v, rd, P.eps, mask, acc);
        group_allreduce<NA>(acc, P.L, lane_in_group, group_in_cta, red, k & 1, mask);
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            float ex = P.goal[0] - p[a][0], ey = P.goal[1] - p[a][1], ez = P.goal[2] - p[a][2];
            float fx, fy, fz;
            if (MOVING || P.apf) { fx = kf[a] * acc.bx[a]; fy = kf[a] * acc.by[a]; fz = kf[a] * acc.bz[a]; }
            else cf_force_static(kf[a], acc.bx[a], acc.by[a], acc.bz[a], v[a][0], v[a][1], v[a][2], fx, fy, fz);
            fx = fmaf(P.k_att, ex, fmaf(-P.k_damp, v[a][0], fx));      // Eq. 6-7
            fy = fmaf(P.k_att, ey, fmaf(-P.k_damp, v[a][1], fy));
            fz = fmaf(P.k_att, ez, fmaf(-P.k_damp, v[a][2], fz));
            if (cost_warp) {
                ca[a].pose(norm3f(ex, ey, ez), acc.dmin[a], P.rcg_is_rd ? rd[a] : P.rcg, P.rco_is_rd ? rd[a] : P.rco);
                if (k >= 2) {                                          // third difference = vf dt^2 (a_k - a_{k-1})
                    float jx = fx - ap[a][0], jy = fy - ap[a][1], jz = fz - ap[a][2];
                    ca[a].add_jerk(fmaf(jx, jx, fmaf(jy, jy, jz * jz)));
                }
                ap[a][0] = fx; ap[a][1] = fy; ap[a][2] = fz;
            }
            v[a][0] = fmaf(P.c_lin, fx, v[a][0]);                      // Eq. 9-10
            v[a][1] = fmaf(P.c_lin, fy, v[a][1]);
            v[a][2] = fmaf(P.c_lin, fz, v[a][2]);
            p[a][0] = fmaf(P.dt, v[a][0], p[a][0]);                    // Eq. 11 (point mass)
            p[a][1] = fmaf(P.dt, v[a][1], p[a][1]);
            p[a][2] = fmaf(P.dt, v[a][2], p[a][2]);
            if (cost_warp) ca[a].add_len(norm3f(v[a][0], v[a][1], v[a][2]));   // |p_new - p| = dt |v|
            if (P.snap_out && k + 1 == P.snap_step && lane_in_group == 0) {
                float* o = P.snap_out + 6 * size_t(gid[a]);
#pragma unroll
                for (int c = 0; c < 3; ++c) { o[c] = p[a][c]; o[3 + c] = v[a][c]; }
            }
            if (P.traj_out && lane_in_group == 0) {
                float* o = P.traj_out + 6 * (size_t(gid[a]) * (P.steps + 1) + k + 1);
#pragma unroll
                for (int c = 0; c < 3; ++c) { o[c] = p[a][c]; o[3 + c] = v[a][c]; }
            }
        }
    }
    // final pose: distance-only pass
    acc.clear();
    sphere_sweep<NA, MOVING, false, false>(sph, svel, P.n_pad, lane_in_group, P.L, fmaf(float(P.steps), P.dt, P.t0), p, v,
                                           rd, P.eps, mask, acc);
    group_allreduce<NA>(acc, P.L, lane_in_group, group_in_cta, red, P.steps & 1, mask);
    if (lane_in_group == 0) {
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            const int i = gid[a];
            ca[a].pose(norm3f(P.goal[0] - p[a][0], P.goal[1] - p[a][1], P.goal[2] - p[a][2]), acc.dmin[a],
                       P.rcg_is_rd ? rd[a] : P.rcg, P.rco_is_rd ? rd[a] : P.rco);
            // sumJ holds sum |f_k - f_{k-1}|^2; a = inv_mass f; third difference = vel_factor dt^2 (a_k - a_{k-1})
            float cj = P.vel_factor * P.dt * P.dt * P.inv_mass;
            ca[a].finish(P, P.dt * ca[a].sumV, cj * cj * ca[a].sumJ, P.cost + 5 * size_t(i));
            P.minclr[i] = ca[a].minclr;
            P.collided[i] = ca[a].collided;
            if (P.agents_out) {
                float* o = P.agents_out + 6 * size_t(i);
#pragma unroll
                for (int c = 0; c < 3; ++c) { o[c] = p[a][c]; o[3 + c] = v[a][c]; }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// 6D pose agents (8-float motor + 6-float body twist), one agent per group
// ---------------------------------------------------------------------------------------------
// The motor's translation is carried as the world vector p = 2 d r^* and its rotor r: the motor product
// M <- M dM is then r <- r r_d, p <- p + R(r) t_d (identical group operation; the additive update keeps
// the FP32 position error at the 3D path's level instead of compounding it through d (x) r_d products).
// The dual part d = (1/2) p (x) r is rebuilt when the state is written out.
struct Pose6 { Quat r; Vec3 p; Vec3 w, nu; };

__device__ __forceinline__ Pose6 load_pose6(const float* s) {
    Pose6 x;
    Quat d = Quat{s[4], s[5], s[6], s[7]};
    x.r = Quat{s[0], s[1], s[2], s[3]};
    x.w = v3(s[8], s[9], s[10]); x.nu = v3(s[11], s[12], s[13]);
    motor_normalise(x.r, d);
    x.p = motor_translation(x.r, d);
    return x;
}

// [n][14] output layout: motor (r, d = (1/2) (0, p) (x) r) + body twist
__device__ __forceinline__ void write_pose6(const Pose6& x, float* o) {
    const Vec3 rv = v3(x.r.x, x.r.y, x.r.z);
    const Vec3 dv = 0.5f * (fma3(x.r.w, x.p, cross(x.p, rv)));
    o[0] = x.r.w; o[1] = x.r.x; o[2] = x.r.y; o[3] = x.r.z;
    o[4] = -0.5f * dot(x.p, rv); o[5] = dv.x; o[6] = dv.y; o[7] = dv.z;
    o[8] = x.w.x; o[9] = x.w.y; o[10] = x.w.z; o[11] = x.nu.x; o[12] = x.nu.y; o[13] = x.nu.z;
}

// body wrench (Eq. 6-8): tau = k_ar e_w - k_dr w;  f = k_att e_v - k_damp nu + R^T f_r
__device__ __forceinline__ void pose6_wrench(const RolloutParams& P, const Pose6& x, Vec3 pos, Quat rg, Vec3 pg,
                                             Vec3 f_r_world, Vec3& tau, Vec3& f) {
    Quat qrel = qmul(qconj(x.r), rg);
    Vec3 trel = qrot_inv(x.r, pg - pos);
    Vec3 ew, ev;
    se3_log_from_quat(qrel, trel, ew, ev);
    Vec3 fb = qrot_inv(x.r, f_r_world);
    tau = fma3(P.k_att_rot, ew, (-P.k_damp_rot) * x.w);
    f = fma3(P.k_att, ev, fma3(-P.k_damp, x.nu, fb));
}

template <bool MOVING, bool CULL>
__device__ __forceinline__ void rollout_pose6(const RolloutParams& P, const float4* sph, const float4* svel,
                                              int agent, int lane_in_group, int group_in_cta, float* red) {
    const unsigned mask = __activemask();
    const int gid = agent_gid(P, agent);
    float rd[1] = {agent_rd(P, gid)};
    const float kf = agent_kf(P, gid);
    const float rcg = P.rcg_is_rd ? rd[0] : P.rcg, rco = P.rco_is_rd ? rd[0] : P.rco;
    agent = gid;
    Pose6 x = load_pose6(P.agents_in + 14 * size_t(agent));
    Quat rg = Quat{P.goal[0], P.goal[1], P.goal[2], P.goal[3]}, dg = Quat{P.goal[4], P.goal[5], P.goal[6], P.goal[7]};
    motor_normalise(rg, dg);
    const Vec3 pg = motor_translation(rg, dg);
    const bool cost_warp = lane_in_group < 32;
    CostAcc ca;
    Vec3 pos = x.p;
    ca.init(norm3f(pg.x - pos.x, pg.y - pos.y, pg.z - pos.z));
    Vec3 dp1 = v3(0, 0, 0), dp2 = v3(0, 0, 0);            // previous two world displacements (Eq. 20)
    StaticAcc<1> acc;
    float p[1][3], v[1][3];
    for (int k = 0; k < P.steps; ++k) {
        const float tk = fmaf(float(k), P.dt, P.t0);
        pos = x.p;
        Vec3 pdot = qrot(x.r, x.nu);                      // world linear velocity of the body origin
        p[0][0] = pos.x; p[0][1] = pos.y; p[0][2] = pos.z;
        v[0][0] = pdot.x; v[0][1] = pdot.y; v[0][2] = pdot.z;
        acc.clear();
        if (P.apf) sphere_sweep<1, MOVING, true, CULL, true>(sph, svel, P.n_pad, lane_in_group, P.L, tk, p, v, rd, P.eps, mask, acc);
        else sphere_sweep<1, MOVING, true, CULL>(sph, svel, P.n_pad, lane_in_group, P.L, tk, p, v, rd, P.eps, mask, acc);
        group_allreduce<1>(acc, P.L, lane_in_group, group_in_cta, red, k & 1, mask);
        Vec3 fr;
        if (MOVING || P.apf) fr = kf * v3(acc.bx[0], acc.by[0], acc.bz[0]);
        else cf_force_static(kf, acc.bx[0], acc.by[0], acc.bz[0], pdot.x, pdot.y, pdot.z, fr.x, fr.y, fr.z);
        if (cost_warp) ca.pose(norm3f(pg.x - pos.x, pg.y - pos.y, pg.z - pos.z), acc.dmin[0], rcg, rco);
        Vec3 tau, f;
        pose6_wrench(P, x, pos, rg, pg, fr, tau, f);
        x.w = fma3(P.c_rot, tau, x.w);                    // Eq. 9-10
        x.nu = fma3(P.c_lin, f, x.nu);
        Quat rd, dd; Vec3 td;
        se3_exp_motor(P.dt * x.w, P.dt * x.nu, rd, dd, td);           // Eq. 11: M <- M exp(dt v)
        Vec3 dp = qrot(x.r, td);                          // world displacement p_new - p
        if (cost_warp) {
            ca.add_len(norm3f(td.x, td.y, td.z));
            if (k >= 2) {
                Vec3 t3 = dp - 2.0f * dp1 + dp2;          // p4 - 3 p3 + 3 p2 - p1 from displacements
                ca.add_jerk(dot(t3, t3));
            }
            dp2 = dp1; dp1 = dp;
        }
        x.p = x.p + dp;
        x.r = qmul(x.r, rd);
        Quat dz = Quat{0, 0, 0, 0};
        motor_normalise(x.r, dz);
        if (P.snap_out && k + 1 == P.snap_step && lane_in_group == 0) write_pose6(x, P.snap_out + 14 * size_t(agent));
        if (P.traj_out && lane_in_group == 0) write_pose6(x, P.traj_out + 14 * (size_t(agent) * (P.steps + 1) + k + 1));
    }
    pos = x.p;
    p[0][0] = pos.x; p[0][1] = pos.y; p[0][2] = pos.z;
    v[0][0] = v[0][1] = v[0][2] = 0.0f;
    acc.clear();
    sphere_sweep<1, MOVING, false, false>(sph, svel, P.n_pad, lane_in_group, P.L, fmaf(float(P.steps), P.dt, P.t0), p, v,
                                          rd, P.eps, mask, acc);
    group_allreduce<1>(acc, P.L, lane_in_group, group_in_cta, red, P.steps & 1, mask);
    if (lane_in_group == 0) {
        ca.pose(norm3f(pg.x - pos.x, pg.y - pos.y, pg.z - pos.z), acc.dmin[0], rcg, rco);
        ca.finish(P, ca.sumV, ca.sumJ, P.cost + 5 * size_t(agent));
        P.minclr[agent] = ca.minclr;
        P.collided[agent] = ca.collided;
        if (P.agents_out) write_pose6(x, P.agents_out + 14 * size_t(agent));
    }
}

// ---------------------------------------------------------------------------------------------
// the persistent rollout kernel: one launch per planning cycle
// ---------------------------------------------------------------------------------------------
template <int KIND, int AT, bool MOVING, bool CULL, int STAGE, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) k_rollout(const __grid_constant__ RolloutParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw);
    float* red = reinterpret_cast<float*>(smem_raw + P.red_off);
    const float4* sph = P.sph;
    const float4* svel = P.svel;
    const int tid = threadIdx.x;
    if (STAGE == 1) {
        float4* tile = reinterpret_cast<float4*>(smem_raw + P.tile_off);
        if (tid == 0) { mbar_init(bar, 1); fence_mbar_init(); }
        __syncthreads();
        if (tid == 0) {
            const uint32_t bytes = uint32_t(P.n_pad) * 16u;
            mbar_arrive_expect_tx(bar, MOVING ? 2u * bytes : bytes);
            const uint32_t chunk = 32768u;
            for (uint32_t o = 0; o < bytes; o += chunk) {
                uint32_t nb = bytes - o < chunk ? bytes - o : chunk;
                tma_bulk_g2s(reinterpret_cast<unsigned char*>(tile) + o,
                             reinterpret_cast<const unsigned char*>(P.sph) + o, nb, bar);
                if (MOVING)
                    tma_bulk_g2s(reinterpret_cast<unsigned char*>(tile) + bytes + o,
                                 reinterpret_cast<const unsigned char*>(P.svel) + o, nb, bar);
            }
        }
        sph = tile;
        svel = tile + P.n_pad;
    }
    const int group_in_cta = tid >> P.logL;
    const int lane_in_group = tid & (P.L - 1);
    const int cta_first = blockIdx.x * P.agents_per_cta;
    int cta_end = cta_first + P.agents_per_cta;
    if (cta_end > P.n_agents) cta_end = P.n_agents;
    const int first = cta_first + group_in_cta * AT;
    int na = cta_end - first;
    if (STAGE == 1) mbar_wait(bar, 0);
    if (na <= 0) return;
    if (KIND == 0) {
        if (AT == 2 && na >= 2) rollout_point3<(AT == 2 ? 2 : 1), MOVING, CULL>(P, sph, svel, first, lane_in_group, group_in_cta, red);
        else rollout_point3<1, MOVING, CULL>(P, sph, svel, first, lane_in_group, group_in_cta, red);
    } else {
        rollout_pose6<MOVING, CULL>(P, sph, svel, first, lane_in_group, group_in_cta, red);
    }
}

// ---------------------------------------------------------------------------------------------
// force query (no integration): warp per agent, spheres from global / L2
// ---------------------------------------------------------------------------------------------
struct ForceParams {
    const float4* sph; const float4* svel; int n_pad;
    const float* agents; int n_agents; int kind;
    float goal[8];
    float k_circ, k_att, k_damp, k_att_rot, k_damp_rot, r_d, eps, t_obs;
    int apf; float inv_rd;
    float* f_rep; float* f_total;
};

template <bool MOVING>
__global__ void __launch_bounds__(256) k_forces(const __grid_constant__ ForceParams P) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (warp >= P.n_agents) return;
    float p[1][3], v[1][3];
    Pose6 x;
    Vec3 pos;
    if (P.kind == 0) {
        const float* s = P.agents + 6 * size_t(warp);
        for (int i = 0; i < 3; ++i) { p[0][i] = s[i]; v[0][i] = s[3 + i]; }
    } else {
        x = load_pose6(P.agents + 14 * size_t(warp));
        pos = x.p;
        Vec3 pdot = qrot(x.r, x.nu);
        p[0][0] = pos.x; p[0][1] = pos.y; p[0][2] = pos.z;
        v[0][0] = pdot.x; v[0][1] = pdot.y; v[0][2] = pdot.z;
    }
    StaticAcc<1> acc;
    acc.clear();
    const float rd[1] = {P.r_d};
    if (P.apf) sphere_sweep<1, MOVING, true, false, true>(P.sph, P.svel, P.n_pad, lane, 32, P.t_obs, p, v, rd, P.eps, 0xffffffffu, acc);
    else sphere_sweep<1, MOVING, true, false>(P.sph, P.svel, P.n_pad, lane, 32, P.t_obs, p, v, rd, P.eps, 0xffffffffu, acc);
    group_allreduce<1>(acc, 32, lane, 0, nullptr, 0, 0xffffffffu);
    Vec3 fr;
    if (MOVING || P.apf) fr = P.k_circ * v3(acc.bx[0], acc.by[0], acc.bz[0]);
    else cf_force_static(P.k_circ, acc.bx[0], acc.by[0], acc.bz[0], v[0][0], v[0][1], v[0][2], fr.x, fr.y, fr.z);
    if (lane != 0) return;
    if (P.f_rep) { float* o = P.f_rep + 3 * size_t(warp); o[0] = fr.x; o[1] = fr.y; o[2] = fr.z; }
    if (P.f_total) {
        if (P.kind == 0) {
            float* o = P.f_total + 3 * size_t(warp);
            for (int i = 0; i < 3; ++i)
                o[i] = fmaf(P.k_att, P.goal[i] - p[0][i], fmaf(-P.k_damp, v[0][i], i == 0 ? fr.x : (i == 1 ? fr.y : fr.z)));
        } else {
            Quat rg = Quat{P.goal[0], P.goal[1], P.goal[2], P.goal[3]}, dg = Quat{P.goal[4], P.goal[5], P.goal[6], P.goal[7]};
            motor_normalise(rg, dg);
            Vec3 pg = motor_translation(rg, dg);
            RolloutParams R{};
            R.k_att = P.k_att; R.k_damp = P.k_damp; R.k_att_rot = P.k_att_rot; R.k_damp_rot = P.k_damp_rot;
            Vec3 tau, f;
            pose6_wrench(R, x, pos, rg, pg, fr, tau, f);
            float* o = P.f_total + 6 * size_t(warp);
            o[0] = tau.x; o[1] = tau.y; o[2] = tau.z; o[3] = f.x; o[4] = f.y; o[5] = f.z;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// selection: lexicographic argmin of (collided, C, index) + hysteresis
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ bool key_less(int ca, float Ca, int ia, int cb, float Cb, int ib) {
    if (ca != cb) return ca < cb;
    if (Ca != Cb) return Ca < Cb;
    return ia < ib;
}
// lane 0 of the reducing warp: hysteresis against the incumbent and the 8-word record (device + pinned host)
__device__ __forceinline__ void selection_record(const float* cost5, const int* collided, int n, float alpha, int prev_best,
                                                 int bi, int bc, float bC, int* out_dev, int* out_host, int seq = 0) {
    int rec[8];
    rec[3] = n > 0 ? bi : -1; rec[4] = n > 0 ? bc : 0; rec[5] = n > 0 ? __float_as_int(bC) : 0x7fc00000;
    rec[6] = 0; rec[7] = 0x7fc00000;
    if (n > 0 && prev_best >= 0 && prev_best < n) {
        float Cp = __ldcg(cost5 + 5 * size_t(prev_best)); int cp = __ldcg(collided + prev_best) ? 1 : 0;
        if (Cp != Cp) { Cp = __int_as_float(0x7f800000); cp = 1; }
        rec[6] = cp; rec[7] = __float_as_int(Cp);
        if (prev_best != bi) {
            const bool improves = (bc < cp) || (bc == cp && bC < alpha * Cp);
            if (!improves) { bi = prev_best; bC = Cp; bc = cp; }
        }
    }
    rec[0] = n > 0 ? bi : -1; rec[1] = n > 0 ? bc : 0; rec[2] = n > 0 ? __float_as_int(bC) : 0x7fc00000;
#pragma unroll
    for (int i = 0; i < 8; ++i) out_dev[i] = rec[i];
    if (out_host) {                                          // pinned host memory: the record, then (ordered behind it) the
#pragma unroll                                                // sequence number the host may be polling for
        for (int i = 0; i < 8; ++i) out_host[i] = rec[i];
        __threadfence_system();
        *reinterpret_cast<volatile int*>(out_host + 8) = seq;
        __threadfence_system();
    }
}
// Tail of a rollout warp: all 32 lanes, converged, after the warp's writer lanes stored the results of `n_done` agents.
// (called from ONE place per kernel, after the group bodies have returned: inlined into every body it perturbed the
// register allocation of the sweep loops, and as a real function call it forced the ABI on the whole kernel)
// Measured on B200 (profiles/r02_selection.md): in the wide 6D kernel the fused tail is free and saves the second launch
// (config 4: 0.418 -> 0.410 ms per cycle).  In the packed point-agent kernels the few extra instructions of the tail
// change ptxas' register assignment of the sweep loops (96-register kernels): config 3's kernel 0.313 -> 0.327 ms, config 1
// 0.041 -> 0.051 ms, 16384 x 4096 9.575 -> 9.647 ms -- more than the ~12 us a selection kernel launched with programmatic
// stream serialisation behind the rollout costs.  So: fused in the wide kernel, a dependent launch after the packed ones.
#ifndef GMAPP_FUSED_SELECT_WIDE
#define GMAPP_FUSED_SELECT_WIDE 1
#endif
#ifndef GMAPP_FUSED_SELECT_X2
#define GMAPP_FUSED_SELECT_X2 0
#endif
template <bool ON>
__device__ __forceinline__ void select_tail(const SelParams& Q, const float* cost5, const int* collided, int n_done, int lane) {
    if (!ON) return;
    if (!Q.ticket) return;
    __threadfence_system();                                  // the writer lanes' results: device-wide, and the final states a
    __syncwarp();                                            // host-buffer cycle wrote to pinned memory, host-visible
    int last = 0;
    if (lane == 0) last = (atomicAdd(Q.ticket, n_done) + n_done == Q.total) ? 1 : 0;
    last = __shfl_sync(0xffffffffu, last, 0);
    if (!last) return;
    __threadfence();
    const int n = Q.total;
    int bc = 2, bi = 0x7fffffff; float bC = __int_as_float(0x7f800000);
    for (int i = lane; i < n; i += 32) {                     // L2 reads: the results were written by other SMs
        float C = __ldcg(cost5 + 5 * size_t(i)); int c = __ldcg(collided + i) ? 1 : 0;
        if (C != C) { C = __int_as_float(0x7f800000); c = 1; }
        if (key_less(c, C, i, bc, bC, bi)) { bc = c; bC = C; bi = i; }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const int oc = __shfl_xor_sync(0xffffffffu, bc, off);
        const float oC = __shfl_xor_sync(0xffffffffu, bC, off);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
        if (key_less(oc, oC, oi, bc, bC, bi)) { bc = oc; bC = oC; bi = oi; }
    }
    if (lane == 0) {
        *Q.ticket = 0;                                       // ready for the next cycle (stream order)
        selection_record(cost5, collided, n, Q.alpha, Q.prev_dev ? *Q.prev_dev : Q.prev, bi, bc, bC, Q.out_dev, Q.out_host, Q.seq);
    }
}

// the same for kernels whose finishing lanes are not whole warps (sub-warp groups, a tuning-only shape): one thread
template <bool ON>
__device__ __forceinline__ void select_tail_serial(const SelParams& Q, const float* cost5, const int* collided, int n_done) {
    if (!ON) return;
    if (!Q.ticket) return;
    __threadfence();
    if (atomicAdd(Q.ticket, n_done) + n_done != Q.total) return;
    __threadfence();
    const int n = Q.total;
    int bc = 2, bi = 0x7fffffff; float bC = __int_as_float(0x7f800000);
    for (int i = 0; i < n; ++i) {
        float C = __ldcg(cost5 + 5 * size_t(i)); int c = __ldcg(collided + i) ? 1 : 0;
        if (C != C) { C = __int_as_float(0x7f800000); c = 1; }
        if (key_less(c, C, i, bc, bC, bi)) { bc = c; bC = C; bi = i; }
    }
    *Q.ticket = 0;
    selection_record(cost5, collided, n, Q.alpha, Q.prev_dev ? *Q.prev_dev : Q.prev, bi, bc, bC, Q.out_dev, Q.out_host, Q.seq);
}

#ifdef GMAPP_MAIN_TU      // non-template kernels: compiled once, in gmapp.cu
// ---------------------------------------------------------------------------------------------
// obstacle packing: (xyz, r) [+ vel] -> float4 arrays, R = r + r_a, sentinel padding to n_cap
// ---------------------------------------------------------------------------------------------
// When `pairs` is given the same launch also writes the sphere-PAIR arrays of the packed kernels (gmapp_rollout_x2.cuh:
// A = (cx0,cx1,cy0,cy1), B = (cz0,cz1,-R0,-R1) [, U, V], `stride` float4 apart): even lanes fetch the odd neighbour's
// sphere by shuffle.  n_cap is even and the block size a multiple of 32, so shuffle partners always exist.
__global__ void k_pack_spheres(const float* __restrict__ xyzr, const float* __restrict__ vel, int n, int n_cap,
                               float r_agent, float4* __restrict__ sph, float4* __restrict__ svel,
                               float4* __restrict__ pairs, int stride) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    // sentinel: far away, never gated, never the minimum
    float4 s = make_float4(kFar, kFar, kFar, 0.0f), u = make_float4(0, 0, 0, 0);
    if (i < n) {
        s = make_float4(xyzr[4 * i], xyzr[4 * i + 1], xyzr[4 * i + 2], xyzr[4 * i + 3] + r_agent);
        if (vel) u = make_float4(vel[3 * i], vel[3 * i + 1], vel[3 * i + 2], 0.0f);
    }
    if (i < n_cap) { sph[i] = s; svel[i] = u; }
    if (!pairs) return;
    float4 t, w;
    t.x = __shfl_down_sync(0xffffffffu, s.x, 1); t.y = __shfl_down_sync(0xffffffffu, s.y, 1);
    t.z = __shfl_down_sync(0xffffffffu, s.z, 1); t.w = __shfl_down_sync(0xffffffffu, s.w, 1);
    w.x = __shfl_down_sync(0xffffffffu, u.x, 1); w.y = __shfl_down_sync(0xffffffffu, u.y, 1);
    w.z = __shfl_down_sync(0xffffffffu, u.z, 1);
    if ((i & 1) || i >= n_cap) return;
    const int j = i >> 1;
    pairs[j] = make_float4(s.x, t.x, s.y, t.y);
    pairs[stride + j] = make_float4(s.z, t.z, -s.w, -t.w);
    if (vel) {
        pairs[2 * stride + j] = make_float4(u.x, w.x, u.y, w.y);
        pairs[3 * stride + j] = make_float4(u.z, w.z, 0.0f, 0.0f);
    }
}

// ---------------------------------------------------------------------------------------------
// selection as a kernel of its own (gmapp_best_agent with another alpha / incumbent than the rollout's tail was armed
// with, and after the kernels that have no fused tail)
// ---------------------------------------------------------------------------------------------
// d_prev (nullable): the incumbent is read from device memory (closed-loop re-planning chains cycles without the host)
__global__ void __launch_bounds__(1024) k_best_agent(const float* __restrict__ cost5, const int* __restrict__ collided,
                                                     int n, float alpha, int prev_best, const int* __restrict__ d_prev,
                                                     int* out_rec, int* host_out, int seq) {
    // launched with programmatic stream serialisation behind the rollout (gmapp_best_agent_ex): wait here for its
    // results; a plain launch returns from this at once
    cudaGridDependencySynchronize();
    if (d_prev) prev_best = *d_prev;
    __shared__ int s_c[32]; __shared__ float s_C[32]; __shared__ int s_i[32];
    int bc = 2, bi = 0x7fffffff; float bC = __int_as_float(0x7f800000);
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        float C = cost5[5 * size_t(i)]; int c = collided[i] ? 1 : 0;
        if (C != C) { C = __int_as_float(0x7f800000); c = 1; }
        if (key_less(c, C, i, bc, bC, bi)) { bc = c; bC = C; bi = i; }
    }
    for (int off = 16; off > 0; off >>= 1) {
        int oc = __shfl_xor_sync(0xffffffffu, bc, off);
        float oC = __shfl_xor_sync(0xffffffffu, bC, off);
        int oi = __shfl_xor_sync(0xffffffffu, bi, off);
        if (key_less(oc, oC, oi, bc, bC, bi)) { bc = oc; bC = oC; bi = oi; }
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { s_c[w] = bc; s_C[w] = bC; s_i[w] = bi; }
    __syncthreads();
    if (w == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        bc = l < nw ? s_c[l] : 2; bC = l < nw ? s_C[l] : __int_as_float(0x7f800000); bi = l < nw ? s_i[l] : 0x7fffffff;
        for (int off = 16; off > 0; off >>= 1) {
            int oc = __shfl_xor_sync(0xffffffffu, bc, off);
            float oC = __shfl_xor_sync(0xffffffffu, bC, off);
            int oi = __shfl_xor_sync(0xffffffffu, bi, off);
            if (key_less(oc, oC, oi, bc, bC, bi)) { bc = oc; bC = oC; bi = oi; }
        }
        if (l == 0) selection_record(cost5, collided, n, alpha, prev_best, bi, bc, bC, out_rec, host_out, seq);
    }
}

// closed-loop re-planning: every agent restarts from the winner's state after exec_steps steps (the snapshot);
// the winner becomes the incumbent; the robot path and the winners are recorded.  w = 6 or 14 floats per state.
__global__ void k_reseed(const float* __restrict__ snap, const int* __restrict__ best_idx, int n, int w, float* agents,
                         int* d_prev, float* path_out, int* best_out, int cycle) {
    const int best = best_idx[0];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n * w) agents[i] = snap[best * w + (i % w)];
    if (i < w && path_out) path_out[cycle * w + i] = snap[best * w + i];
    if (i == 0) { *d_prev = best; if (best_out) best_out[cycle] = best; }
}

#endif  // GMAPP_MAIN_TU

// ---------------------------------------------------------------------------------------------
// FP32 peak microkernel: 8 independent FMA chains per thread, register only
// ---------------------------------------------------------------------------------------------
template <bool X2>
__global__ void __launch_bounds__(256) k_fma_peak(float* out, int iters, float a, float b) {
    float x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = float(threadIdx.x + i) * 1e-3f;
    if (X2) {
        unsigned long long X[8], A, Bv;
        asm("mov.b64 %0, {%1, %2};" : "=l"(A) : "f"(a), "f"(a));
        asm("mov.b64 %0, {%1, %2};" : "=l"(Bv) : "f"(b), "f"(b));
#pragma unroll
        for (int i = 0; i < 8; ++i) asm("mov.b64 %0, {%1, %2};" : "=l"(X[i]) : "f"(x[2 * i]), "f"(x[2 * i + 1]));
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int i = 0; i < 8; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(X[i]) : "l"(A), "l"(Bv));
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) asm("mov.b64 {%0, %1}, %2;" : "=f"(x[2 * i]), "=f"(x[2 * i + 1]) : "l"(X[i]));
    } else {
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], a, b);
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == 123.456f) out[0] = s;      // never true in practice; keeps the chains alive
}

}  // namespace gmapp
