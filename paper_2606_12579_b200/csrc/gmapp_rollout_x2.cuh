// gmapp_rollout_x2.cuh -- the packed-FP32 rollout kernel for 3D point agents over static or (template flag MV) moving
// spheres (sm_100a); its sweep, reduction and hand-over pieces are reused by gmapp_rollout_wide.cuh (6D agents).
//
// Same method as gmapp_kernels.cuh (Eq. 2-3, 6-11, 16-20 of the paper), different machine mapping:
//
//  * Packed FP32 math.  Spheres are stored as PAIRS, A[j] = (cx0,cx1, cy0,cy1), B[j] = (cz0,cz1, -R0,-R1)
//    (R = r_j + r_a), so one LDS.128 pair feeds fma.rn.f32x2 / add.f32x2 / mul.f32x2 (SASS FFMA2 / FADD2 /
//    FMUL2: one issue slot for two pairs).  The agent state is the broadcast operand.  MUFU.RSQ / MUFU.RCP,
//    the clamp, the gate and q - t^2 (needs a negated operand) stay scalar.  The gate is a predicated
//    MUFU.RCP into a zeroed register, so a pair outside r_d contributes exactly 0.
//  * A group of L lanes owns NA (1 or 2) agents; lane l sweeps sphere pairs l, l+L, ...  The 3 NA partial
//    sums are combined by a TRANSPOSED xor-butterfly (each step halves the number of live values: 8 SHFL
//    for 6 values instead of 30), the clearance minimum by one REDUX.MIN on an order-preserving integer
//    key.  Fixed order, no atomics: bit-reproducible.
//  * When a group spans several warps (L >= 64) its W = L/32 sweep warps post their partial sums to shared
//    memory and a dedicated EPILOGUE WARP of the group adds them, integrates BOTH agents at once (agent a on
//    lanes 0-15, agent b on lanes 16-31), publishes the new state and only then accumulates the costs; the
//    sweep warps pick the state up after a named barrier.  Split arrive / sync barriers and parity double-
//    buffering: one round trip per step; what does not need the sums is computed before the wait.
//  * Two-pass distance refinement: force sweeps run on the raw MUFU.RSQ distance; only a warp one of whose lanes came
//    within R/16 of a surface repeats its sweep with the Newton step (and stays refined while its agents are near).
//  * With more than 32 agents per CTA every warp owns a block of agents and walks it in chunks of two inside each
//    step (per-agent state records in shared memory): no cross-warp traffic at all, 0.63 of FP32 peak.
//  * Template parameters where a run-time choice costs speed: CULL (warp-vote skip of the force half), STAGE (shared
//    memory vs L2), APF (Eq. 1 instead of Eq. 2-3), per-agent detection radii (PER), and XT, the snapshot /
//    trajectory stores of gmapp_replan / gmapp_set_trajectory_output.
//
// Shares nothing with oracle/.
#pragma once
#include "gmapp_kernels.cuh"

namespace gmapp {

typedef unsigned long long u64;

#ifndef GMAPP_X2_UNROLL
#define GMAPP_X2_UNROLL 4      // sphere-pair iterations unrolled in the sweep (measured best on B200)
#endif
constexpr int kX2Unroll = GMAPP_X2_UNROLL;
#ifndef GMAPP_X2_HALF_INT
#define GMAPP_X2_HALF_INT 0
#endif

__device__ __forceinline__ u64 pk2(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk2(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 bc2(float x) { return pk2(x, x); }      // ptxas folds this into the .F32 broadcast operand form
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ float min3f(float a, float b, float c) { float y; asm("min.f32 %0, %1, %2, %3;" : "=f"(y) : "f"(a), "f"(b), "f"(c)); return y; }
__device__ __forceinline__ void named_bar_arrive(int id, int count) {
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory");
}
// order-preserving float <-> int key (an involution): integer order of the keys = float order of the values
__device__ __forceinline__ int fkey(float x) { int b = __float_as_int(x); return b ^ ((b >> 31) & 0x7fffffff); }
__device__ __forceinline__ float fkey_inv(int k) { return __int_as_float(k ^ ((k >> 31) & 0x7fffffff)); }

// One MUFU.RCP per sphere PAIR in the circular-field sweep (static spheres): r = 1 / (K n0 n1) with n = d_O |d|^2,
// 1/(K n0) = r n1 and 1/n1 = r (K n0).  K = 2^47 centres the product of two denominators (each between ~1e-33, an agent
// exactly on a sphere centre, and ~1e26, a sphere 1e8 m away) in the FP32 range.  The low half of every accumulator
// therefore holds its sum divided by K; acc_fold() puts the two halves together.  Sentinel pairs sit at kFar (finite
// denominators: 0 * inf would poison the real sphere sharing a pair with a sentinel).
#ifndef GMAPP_X2_PAIR_RCP
#define GMAPP_X2_PAIR_RCP 0
#endif
constexpr float kPairK = 140737488355328.0f;               // 2^47
template <bool SCALED> __device__ __forceinline__ float acc_fold(u64 v) {
    float lo, hi; upk2(v, lo, hi);
    return SCALED ? fmaf(lo, kPairK, hi) : lo + hi;
}
template <bool APF, bool MV> __host__ __device__ constexpr bool acc_scaled() { return GMAPP_X2_PAIR_RCP && !APF && !MV; }

struct RolloutX2Params {
    const float4* pairA;      // [n2p] (cx0,cx1,cy0,cy1)
    const float4* pairB;      // [n2p] (cz0,cz1,-R0,-R1)
    int n2p;                  // sphere pairs, padded to a multiple of L with sentinels
    const float* agents_in;   // [n][6]
    float* agents_out;        // [n][6] or nullptr
    int n_agents, agents_per_cta;
    int L, logL;
    int steps;
    float goal[3];
    float dt;
    float k_circ, k_att, k_damp;
    float c_lin;              // vel_factor * dt * inv_mass   (Eq. 9-10)
    float inv_mass, vel_factor;
    float r_d, eps;
    float rcg, rco;           // Eq. 17 / 18 radii
    float w_goal, w_obs, w_path, w_smooth, a_max;
    float* cost;              // [n][5]
    float* minclr;            // [n]
    int* collided;            // [n]
    int tile_off;             // byte offset of the sphere tile in dynamic shared memory
    int xch_off;              // byte offset of the cross-warp exchange area
    int rec_off;              // byte offset of the per-agent state records (mode 4)
    int stage;                // 1: sphere pairs staged in shared memory by TMA bulk copies; 0: read through L1/L2
    float t0;                 // moving spheres: obstacles are evaluated at t0 + k dt (pair arrays U, V behind A, B)
    int apf;                  // 1: APF heuristic (Eq. 1) instead of the circular field (Eq. 2-3)
    // heterogeneous ensemble (gmapp_set_agent_params): all nullable
    const int* agent_idx;     // [n_agents] this launch's agents as indices into the caller's arrays (one launch per heuristic)
    const float* rd_arr;      // per-agent detection radius r_d, indexed by the caller's agent index
    const float* kf_arr;      // per-agent gain k_f
    int rcg_is_rd, rco_is_rd; // Eq. 17 / 18 radii default to the agent's own r_d
    float* snap_out;          // closed-loop re-planning: [n][6] states after snap_step steps, or nullptr
    int snap_step;            // 1..steps
    float* traj_out;          // nullable: [n][steps+1][6] every pose of every agent (pose 0 = start state, written by the host side)
    const int* count_dev;     // nullable: device-resident sphere count of a built sphere world (gmapp_build_sphere_world);
    int n_cap;                // the kernel then sweeps only the pairs that hold real spheres (the slots behind are sentinels)
    // TMA tile ring (STAGE == 2: sphere sets beyond shared memory)
    int ring_tp;              // sphere pairs per tile (a multiple of L)
    int ring_off;             // byte offset of the ring's mbarriers (full[kRingStages], empty[kRingStages])
    const float* sph_stats;   // device: {largest R = r_j + r_a, largest sphere speed |u_j|} of the sphere world
    SelParams sel;            // selection fused into the rollout's tail (gmapp_kernels.cuh)
};

__device__ __forceinline__ int agent_gid(const RolloutX2Params& P, int i) { return P.agent_idx ? P.agent_idx[i] : i; }
__device__ __forceinline__ float agent_rd(const RolloutX2Params& P, int gid) { return P.rd_arr ? P.rd_arr[gid] : P.r_d; }

// Detection radius seen by the sweeps: PER = false -> the uniform r_d of the launch (a kernel parameter, so it stays
// in a uniform register and costs no vector-register read in the gate compare); PER = true -> per-agent values
// (gmapp_set_agent_params).  Chosen once per kernel by a top-level branch, not inside the loops.
template <int NA, bool PER>
struct RdSel {
    float v[NA];
    float u;
    __device__ __forceinline__ float get(int a) const { return PER ? v[a] : u; }
};

// per-lane partial sums of NA agents over the lane's sphere pairs (both halves of a pair kept apart)
template <int NA>
struct X2Acc {
    u64 bx[NA], by[NA], bz[NA];
    float dmin[NA];
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int a = 0; a < NA; ++a) { bx[a] = by[a] = bz[a] = 0ull; dmin[a] = __int_as_float(0x7f800000); }
    }
};

// Stage-major sweep over U trips at once (circular field, static spheres, branch-free).  ptxas keeps unrolled trips
// strictly one after another (it only interleaves what the SOURCE writes stage by stage, as the NA agents of a trip), and
// a warp issues in order: with one trip at a time a warp has NA packed chains in flight and exposes the MUFU.RSQ -> FMA ->
// MUFU.RCP -> FMA latency of every trip.  Written stage by stage over K = NA x U (agent, trip) slots, two trips' chains
// overlap inside the warp.  Same arithmetic per pair, same order of accumulation per lane (trip u before trip u + 1).
#ifndef GMAPP_X2_U
#define GMAPP_X2_U 1
#endif
// Group widths as compile-time constants where the common shapes have them (128 lanes: config 3 and the 1024-agent sweep rows;
// 64 / 128 in the mixed-width mode): the unrolled trips then address the tile with immediate offsets instead of one LEA per
// array and trip -- 0.75 issue cycles of 44 per agent-trip (config 3: 0.3130 -> 0.3060 ms).
#ifndef GMAPP_X2_L128
#define GMAPP_X2_L128 1
#endif
#ifndef GMAPP_X2_U_UNROLL
#define GMAPP_X2_U_UNROLL 2
#endif
constexpr int kX2UUnroll = GMAPP_X2_U_UNROLL;
template <int NA, int U, class RD, bool REFINE>
__device__ __forceinline__ void sweep_x2_cf_u(const float4* __restrict__ tA, const float4* __restrict__ tB, int iters,
                                              int j0, int L, const float (&p)[NA][3], const float (&v)[NA][3],
                                              const RD& rd, float eps, X2Acc<NA>& acc) {
    constexpr int K = NA * U;
    const u64 tiny = bc2(kTiny), half = bc2(0.5f);
#pragma unroll kX2UUnroll
    for (int i = 0, j = j0; i < iters; ++i, j += U * L) {
        u64 cx[U], cy[U], cz[U], nR[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const float4 s0 = tA[j + u * L], s1 = tB[j + u * L];
            cx[u] = pk2(s0.x, s0.y); cy[u] = pk2(s0.z, s0.w); cz[u] = pk2(s1.x, s1.y); nR[u] = pk2(s1.z, s1.w);
        }
        u64 dx[K], dy[K], dz[K], q[K], y[K];
        float d0[K], d1[K];
#pragma unroll
        for (int k = 0; k < K; ++k) {                          // stage 1: d, |d|^2
            const int a = k % NA, u = k / NA;
            dx[k] = sub2(cx[u], bc2(p[a][0])); dy[k] = sub2(cy[u], bc2(p[a][1])); dz[k] = sub2(cz[u], bc2(p[a][2]));
            q[k] = fma2(dx[k], dx[k], fma2(dy[k], dy[k], fma2(dz[k], dz[k], tiny)));
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {                          // stage 2: MUFU.RSQ
            float q0, q1; upk2(q[k], q0, q1);
            y[k] = pk2(rsqrt_approx(q0), rsqrt_approx(q1));
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {                          // stage 3: surface distance, clearance minimum
            const int a = k % NA, u = k / NA;
            u64 ds;
            if (!REFINE) ds = fma2(q[k], y[k], nR[u]);
            if (REFINE) {
                const u64 t = mul2(q[k], y[k]);
                ds = add2(t, nR[u]);
                const u64 hy = mul2(y[k], half);
                float t0, t1, q0, q1; upk2(t, t0, t1); upk2(q[k], q0, q1);
                const u64 e = pk2(fmaf(-t0, t0, q0), fmaf(-t1, t1, q1));
                ds = fma2(hy, e, ds);
            }
            upk2(ds, d0[k], d1[k]);
            acc.dmin[a] = min3f(acc.dmin[a], d0[k], d1[k]);
        }
        u64 rr[K];
#pragma unroll
        for (int k = 0; k < K; ++k) {                          // stage 4: gate, clamp, MUFU.RCP
            const int a = k % NA;
            const u64 den = mul2(pk2(fmaxf(d0[k], eps), fmaxf(d1[k], eps)), q[k]);
            float n0, n1; upk2(den, n0, n1);
            float r0 = 0.0f, r1 = 0.0f;
            if (d0[k] <= rd.get(a)) r0 = rcp_approx(n0);
            if (d1[k] <= rd.get(a)) r1 = rcp_approx(n1);
            rr[k] = pk2(r0, r1);
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {                          // stage 5: s = d.v, w, accumulate
            const int a = k % NA;
            const u64 s = fma2(dx[k], bc2(v[a][0]), fma2(dy[k], bc2(v[a][1]), mul2(dz[k], bc2(v[a][2]))));
            const u64 w = mul2(s, rr[k]);
            acc.bx[a] = fma2(w, dx[k], acc.bx[a]);
            acc.by[a] = fma2(w, dy[k], acc.by[a]);
            acc.bz[a] = fma2(w, dz[k], acc.bz[a]);
        }
    }
}

// One lane's slice of the sphere sum: pairs lane, lane+L, ... ; FORCE=false is the distance-only final pass.
// APF = true: Eq. 1 in the Khatib form on the clamped surface distance (reading N1),
// f_j = -k_f (1/d_O - 1/r_d) / d_O^2 * d/|d|; the sums then hold the force itself (no velocity factor).
template <int NA, bool FORCE, bool CULL, bool APF = false, class RD = RdSel<NA, false>, bool REFINE = true>
__device__ __forceinline__ void sweep_x2(const float4* __restrict__ tA, const float4* __restrict__ tB, int trips,
                                         int lane, int L, const float (&p)[NA][3], const float (&v)[NA][3],
                                         const RD& rd, float eps, unsigned mask, X2Acc<NA>& acc) {
    const u64 tiny = bc2(kTiny), half = bc2(0.5f);
    int i_first = 0;
    if (GMAPP_X2_U > 1 && FORCE && !CULL && !APF && !GMAPP_X2_PAIR_RCP) {     // U trips at once, stage by stage; the tail below
        const int iters = trips / GMAPP_X2_U;
        sweep_x2_cf_u<NA, GMAPP_X2_U, RD, REFINE>(tA, tB, iters, lane, L, p, v, rd, eps, acc);
        i_first = iters * GMAPP_X2_U;
    }
#pragma unroll kX2Unroll
    for (int i = i_first, j = lane + i_first * L; i < trips; ++i, j += L) {
        const float4 s0 = tA[j], s1 = tB[j];
        const u64 cx = pk2(s0.x, s0.y), cy = pk2(s0.z, s0.w), cz = pk2(s1.x, s1.y), nR = pk2(s1.z, s1.w);
        u64 dx[NA], dy[NA], dz[NA], q[NA], yy[NA];
        float d0[NA], d1[NA];
        bool any = false;
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            dx[a] = sub2(cx, bc2(p[a][0])); dy[a] = sub2(cy, bc2(p[a][1])); dz[a] = sub2(cz, bc2(p[a][2]));
            q[a] = fma2(dx[a], dx[a], fma2(dy[a], dy[a], fma2(dz[a], dz[a], tiny)));
            float q0, q1; upk2(q[a], q0, q1);
            const float y0 = rsqrt_approx(q0), y1 = rsqrt_approx(q1);
            const u64 y = pk2(y0, y1);
            yy[a] = y;
            u64 ds;
            if (!REFINE) ds = fma2(q[a], y, nR);                         // dist - R from the raw MUFU.RSQ (~1.9e-7 relative in dist), one FFMA2
            if (REFINE) {
                const u64 t = mul2(q[a], y);
                ds = add2(t, nR);
                const u64 hy = mul2(y, half);
                float t0, t1; upk2(t, t0, t1);
                const u64 e = pk2(fmaf(-t0, t0, q0), fmaf(-t1, t1, q1)); // Newton residual q - t^2 (exact in the FMA)
                ds = fma2(hy, e, ds);                                    // dist - R, dist to ~1 ulp
            }
            upk2(ds, d0[a], d1[a]);
            acc.dmin[a] = min3f(acc.dmin[a], d0[a], d1[a]);
            if (CULL) any = any || (fminf(d0[a], d1[a]) <= rd.get(a));
        }
        if (!FORCE) continue;
        if (CULL) { if (!__any_sync(mask, any)) continue; }
        if (APF) {
#pragma unroll
            for (int a = 0; a < NA; ++a) {
                float r0 = 0.0f, r1 = 0.0f;                                  // 1/d_O inside r_d, else 0 (contributes exactly 0)
                if (d0[a] <= rd.get(a)) r0 = rcp_approx(fmaxf(d0[a], eps));
                if (d1[a] <= rd.get(a)) r1 = rcp_approx(fmaxf(d1[a], eps));
                const u64 ro = pk2(r0, r1);
                const u64 m = mul2(mul2(sub2(bc2(rcp_approx(rd.get(a))), ro), mul2(ro, ro)), yy[a]);   // -(1/d_O - 1/r_d)/d_O^2 / |d|
                acc.bx[a] = fma2(m, dx[a], acc.bx[a]);
                acc.by[a] = fma2(m, dy[a], acc.by[a]);
                acc.bz[a] = fma2(m, dz[a], acc.bz[a]);
            }
            continue;
        }
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            const u64 den = mul2(pk2(fmaxf(d0[a], eps), fmaxf(d1[a], eps)), q[a]);     // d_O * |d|^2
            float n0, n1; upk2(den, n0, n1);
            float r0 = 0.0f, r1 = 0.0f;
#if GMAPP_X2_PAIR_RCP
            const float n0k = n0 * kPairK;
            const float r = rcp_approx(n0k * n1);                            // one MUFU.RCP for the two pairs
            if (d0[a] <= rd.get(a)) r0 = r * n1;                             // 1 / (K n0); Alg. 1 line 7: outside r_d contributes 0
            if (d1[a] <= rd.get(a)) r1 = r * n0k;                            // 1 / n1
#else
            if (d0[a] <= rd.get(a)) r0 = rcp_approx(n0);                     // Alg. 1 line 7: outside r_d contributes 0
            if (d1[a] <= rd.get(a)) r1 = rcp_approx(n1);
#endif
            const u64 s = fma2(dx[a], bc2(v[a][0]), fma2(dy[a], bc2(v[a][1]), mul2(dz[a], bc2(v[a][2]))));
            const u64 w = mul2(s, pk2(r0, r1));
            acc.bx[a] = fma2(w, dx[a], acc.bx[a]);
            acc.by[a] = fma2(w, dy[a], acc.by[a]);
            acc.bz[a] = fma2(w, dz[a], acc.bz[a]);
        }
    }
}

// each 16-lane half of the warp sums its own (x, y, z) over its lanes; every lane of a half gets the three sums.
// Transposed butterfly: step 8 leaves (x, y) on the lanes with bit 3 clear and z on the others, step 4 one value
// per lane, steps 2 and 1 finish: 5 shuffles + 3 to hand the sums round.
__device__ __forceinline__ void half_sum3(float kx, float ky, float kz, int lane, float& X, float& Y, float& Z) {
    const unsigned full = 0xffffffffu;
    const bool h8 = lane & 8, h4 = lane & 4;
    float r1 = __shfl_xor_sync(full, h8 ? kx : kz, 8);
    float r2 = __shfl_xor_sync(full, ky, 8);
    if (h8) kz += r1; else { kx += r1; ky += r2; }
    float send = h8 ? kz : (h4 ? kx : ky);
    float keep = h8 ? kz : (h4 ? ky : kx);
    float u = keep + __shfl_xor_sync(full, send, 4);
    u += __shfl_xor_sync(full, u, 2);
    u += __shfl_xor_sync(full, u, 1);
    const int base = lane & 16;
    X = __shfl_sync(full, u, base); Y = __shfl_sync(full, u, base | 4); Z = __shfl_sync(full, u, base | 8);
}

// ---------------------------------------------------------------------------------------------
// packed f32x2 sweep for MOVING spheres.  Sphere pairs: A = (cx0,cx1,cy0,cy1), B = (cz0,cz1,-R0,-R1) at t = 0,
// U = (ux0,ux1,uy0,uy1), V = (uz0,uz1,0,0).  Per pair (reading G5/G25): c(t) = c + t u, v_rel = v - u,
// f_j = w [ (s/|v_rel|) v_rel - |v_rel| d ],  w = s / (d_O |d|^2),  s = d.v_rel, accumulated directly
// (k_f applied after the sum).  The distance half is the static one.
// ---------------------------------------------------------------------------------------------
template <int NA, bool FORCE, bool CULL, bool APF = false, class RD = RdSel<NA, false>, bool REFINE = true>
__device__ __forceinline__ void sweep_x2_moving(const float4* __restrict__ tA, const float4* __restrict__ tB,
                                                const float4* __restrict__ tU, const float4* __restrict__ tV, int trips,
                                                int lane, int L, float tk, const float (&p)[NA][3], const float (&v)[NA][3],
                                                const RD& rd, float eps, unsigned mask, X2Acc<NA>& acc) {
    const u64 tiny = bc2(kTiny), half = bc2(0.5f), t2 = bc2(tk);
#pragma unroll 2
    for (int i = 0, j = lane; i < trips; ++i, j += L) {
        const float4 s0 = tA[j], s1 = tB[j], s2 = tU[j], s3 = tV[j];
        const u64 ux = pk2(s2.x, s2.y), uy = pk2(s2.z, s2.w), uz = pk2(s3.x, s3.y), nR = pk2(s1.z, s1.w);
        const u64 cx = fma2(ux, t2, pk2(s0.x, s0.y)), cy = fma2(uy, t2, pk2(s0.z, s0.w)), cz = fma2(uz, t2, pk2(s1.x, s1.y));
        u64 dx[NA], dy[NA], dz[NA], q[NA], yy[NA];
        float d0[NA], d1[NA];
        bool any = false;
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            dx[a] = sub2(cx, bc2(p[a][0])); dy[a] = sub2(cy, bc2(p[a][1])); dz[a] = sub2(cz, bc2(p[a][2]));
            q[a] = fma2(dx[a], dx[a], fma2(dy[a], dy[a], fma2(dz[a], dz[a], tiny)));
            float q0, q1; upk2(q[a], q0, q1);
            const u64 y = pk2(rsqrt_approx(q0), rsqrt_approx(q1));
            yy[a] = y;
            u64 ds;
            if (!REFINE) ds = fma2(q[a], y, nR);
            if (REFINE) {
                const u64 t = mul2(q[a], y);
                ds = add2(t, nR);
                const u64 hy = mul2(y, half);
                float t0, t1; upk2(t, t0, t1);
                const u64 e = pk2(fmaf(-t0, t0, q0), fmaf(-t1, t1, q1));
                ds = fma2(hy, e, ds);
            }
            upk2(ds, d0[a], d1[a]);
            acc.dmin[a] = min3f(acc.dmin[a], d0[a], d1[a]);
            if (CULL) any = any || (fminf(d0[a], d1[a]) <= rd.get(a));
        }
        if (!FORCE) continue;
        if (CULL) { if (!__any_sync(mask, any)) continue; }
        if (APF) {                                          // Eq. 1 depends on positions only
#pragma unroll
            for (int a = 0; a < NA; ++a) {
                float r0 = 0.0f, r1 = 0.0f;
                if (d0[a] <= rd.get(a)) r0 = rcp_approx(fmaxf(d0[a], eps));
                if (d1[a] <= rd.get(a)) r1 = rcp_approx(fmaxf(d1[a], eps));
                const u64 ro = pk2(r0, r1);
                const u64 m = mul2(mul2(sub2(bc2(rcp_approx(rd.get(a))), ro), mul2(ro, ro)), yy[a]);
                acc.bx[a] = fma2(m, dx[a], acc.bx[a]);
                acc.by[a] = fma2(m, dy[a], acc.by[a]);
                acc.bz[a] = fma2(m, dz[a], acc.bz[a]);
            }
            continue;
        }
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            const u64 vx = sub2(bc2(v[a][0]), ux), vy = sub2(bc2(v[a][1]), uy), vz = sub2(bc2(v[a][2]), uz);
            const u64 n2 = fma2(vx, vx, fma2(vy, vy, fma2(vz, vz, tiny)));
            float m0, m1; upk2(n2, m0, m1);
            const float i0 = rsqrt_approx(m0), i1 = rsqrt_approx(m1);
            const u64 inv = pk2(i0, i1), ninv = pk2(-i0, -i1);
            const u64 nvn = mul2(n2, ninv);                                              // -|v_rel|
            const u64 den = mul2(pk2(fmaxf(d0[a], eps), fmaxf(d1[a], eps)), q[a]);
            float n0, n1; upk2(den, n0, n1);
            float r0 = 0.0f, r1 = 0.0f;
            if (d0[a] <= rd.get(a)) r0 = rcp_approx(n0);
            if (d1[a] <= rd.get(a)) r1 = rcp_approx(n1);
            const u64 s = fma2(dx[a], vx, fma2(dy[a], vy, mul2(dz[a], vz)));
            const u64 w = mul2(s, pk2(r0, r1));
            const u64 c1 = mul2(mul2(w, s), inv), c2 = mul2(w, nvn);
            acc.bx[a] = fma2(c1, vx, fma2(c2, dx[a], acc.bx[a]));
            acc.by[a] = fma2(c1, vy, fma2(c2, dy[a], acc.by[a]));
            acc.bz[a] = fma2(c1, vz, fma2(c2, dz[a], acc.bz[a]));
        }
    }
}

// Two-pass distance refinement.  The Newton step on MUFU.RSQ (5 of the ~19 FP32 lane-operations per pair) only matters
// where an agent is close to a surface: the raw distance is off by <= 1.9e-7 |d|, i.e. the surface distance d_O by a
// relative 1.9e-7 (1 + R/d_O), which stays below 3.3e-6 (CF; the force is ~ 1/d_O) or 3.4e-6 (APF, ~ 1/d_O^3) while
// d_O >= R / kNearK.  So a force sweep first runs WITHOUT the refinement and tracks the clearance as always; only if some
// lane of the warp came closer than thr = (largest R among the lane's own spheres) / kNearK to any of them is the sweep of
// that warp and step repeated WITH it.  Agents of a circular field hug surfaces for many steps, so a warp that had to
// repeat stays in the refined mode (`hot`, one pass per step, the cost of the always-refined kernel) until its agents
// are clear again; the decision is a function of the trajectory only, so results stay bit-reproducible.  The
// distance-only final pass and the collision decision it feeds always refine.  Not part of the 35 algorithmic flop per pair either way.
#ifndef GMAPP_X2_TWO_PASS
#define GMAPP_X2_TWO_PASS 1
#endif
template <bool APF> __device__ __forceinline__ float near_k() { return APF ? 5.0f : 16.0f; }

// thr of this lane: its spheres are the same every step (pairs lane, lane + L, ...), so this runs once per rollout
template <bool APF>
__device__ __forceinline__ float lane_near_thr(const float4* __restrict__ tB, int trips, int lane, int L) {
    float m = 0.0f;                                        // min of -R
    for (int i = 0, j = lane; i < trips; ++i, j += L) { const float4 s = tB[j]; m = fminf(m, fminf(s.z, s.w)); }
    return -m / near_k<APF>();
}

// One entry point for both sweeps.  The pair arrays sit at equal distances: B = A + d, U = A + 2 d, V = A + 3 d.
template <int NA, bool FORCE, bool CULL, bool APF, bool MV, bool REFINE, class RD>
__device__ __forceinline__ void sweep_pass(const float4* __restrict__ tA, const float4* __restrict__ tB, int trips, int lane, int L,
                                           float tk, const float (&p)[NA][3], const float (&v)[NA][3], const RD& rd, float eps,
                                           unsigned mask, X2Acc<NA>& acc) {
    if (MV) sweep_x2_moving<NA, FORCE, CULL, APF, RD, REFINE>(tA, tB, tB + (tB - tA), tB + 2 * (tB - tA), trips, lane, L, tk, p, v, rd, eps, mask, acc);
    else    sweep_x2<NA, FORCE, CULL, APF, RD, REFINE>(tA, tB, trips, lane, L, p, v, rd, eps, mask, acc);
}
template <int NA, bool FORCE, bool CULL, bool APF, bool MV, class RD>
__device__ __forceinline__ void sweep_any(const float4* __restrict__ tA, const float4* __restrict__ tB, int trips, int lane, int L,
                                          float tk, const float (&p)[NA][3], const float (&v)[NA][3], const RD& rd, float eps,
                                          unsigned mask, float thr, bool& hot, X2Acc<NA>& acc) {
    if (FORCE && GMAPP_X2_TWO_PASS) {
        bool near = false;
        if (!hot) {
            sweep_pass<NA, FORCE, CULL, APF, MV, false>(tA, tB, trips, lane, L, tk, p, v, rd, eps, mask, acc);
#pragma unroll
            for (int a = 0; a < NA; ++a) near = near || (acc.dmin[a] < thr);
            if (!__any_sync(mask, near)) return;
            acc.clear();                                   // came close: this sweep again, refined, and stay refined
        }
        sweep_pass<NA, FORCE, CULL, APF, MV, true>(tA, tB, trips, lane, L, tk, p, v, rd, eps, mask, acc);
        near = false;
#pragma unroll
        for (int a = 0; a < NA; ++a) near = near || (acc.dmin[a] < thr);
        hot = __any_sync(mask, near);                      // back to the raw distance once the warp's agents are clear again
        return;
    }
    sweep_pass<NA, FORCE, CULL, APF, MV, true>(tA, tB, trips, lane, L, tk, p, v, rd, eps, mask, acc);
}

// ---------------------------------------------------------------------------------------------
// TMA tile ring (STAGE == 2): sphere sets that do not fit shared memory (config 5 at 16384 / 65536 spheres).
// The pair arrays are cut into tiles of `tp` pairs, streamed from L2 into a ring of kRingStages shared-memory slots by
// 1-D TMA bulk copies.  Per slot: an mbarrier full[s] (count 1 + transaction bytes: "the tile has landed") and a
// release counter done[s].  Every consumer warp of the CTA walks the SAME tile sequence -- (steps + 1) passes x `rounds`
// x tiles -- so one copy of a tile serves all agents of the CTA (a warp with fewer agent chunks than the others still
// visits, and releases, the tiles of the rounds it skips).  There is no producer warp (a 21st warp would cut the
// register budget of the 20-warp CTA from 96 to 80) and nobody ever waits for a slot to drain: the warp that releases a
// slot LAST (its atomic increment of done[s] reaches the number of consumer warps) refills it on the spot with the
// tile kRingStages visits ahead.  Warps may drift apart by up to kRingStages - 1 tiles, which keeps one group's reduce /
// integrate round trip overlapped with the other groups' sweeps.
// Distance refinement in ring mode is PREDICTED instead of repeated (a warp cannot go back to tiles that have left the
// ring): a lane's clearance minimum m over its own spheres at pose k bounds the same minimum at pose k + 1 from below by
// m - dt (|v| + max |u_j|) (v: the new velocity, Eq. 11), so the warp sweeps step k + 1 on the raw MUFU.RSQ distance
// only if that bound is >= thr = (largest R among the lane's spheres) / kNearK on all its lanes (then every pair has
// d_O >= R_j / kNearK, the condition of the two-pass scheme above); step 0 and the final pass always refine.  Same
// granularity as the two-pass scheme: only the warps whose own spheres are close pay for the Newton step.
// ---------------------------------------------------------------------------------------------
constexpr int kRingStages = 3;
struct RingView {
    uint64_t* full;           // [kRingStages]
    int* done;                // [kRingStages] consumer warps that have released the slot's current tile
    const float4* slots;      // slot s at slots + s * slot_f4; inside a slot the arrays A, B (, U, V) are tp float4 apart
    int tp, slot_f4, nt, last_pairs, narr, consumers, total;
};
struct RingPos {
    int slot; uint32_t parity;
    int t, v;                 // tile index inside the pass, visit index
    __device__ __forceinline__ void advance(int nt) {
        if (++slot == kRingStages) { slot = 0; parity ^= 1u; }
        if (++t == nt) t = 0;
        ++v;
    }
};
struct SphSrc {               // where a sweep finds the sphere pairs: resident arrays (STAGE 0 / 1) or the ring
    const float4* tA; const float4* tB; int n2p;
    RingView ring; RingPos pos;
    float umax_dt;            // ring mode: dt * (largest sphere speed)
};

// one elected thread: copy tile t of the pair arrays into `slot` (completion on full[slot])
__device__ __forceinline__ void ring_issue(const RolloutX2Params& P, const RingView& R, int t, int slot) {
    const uint32_t pairs = t == R.nt - 1 ? uint32_t(R.last_pairs) : uint32_t(R.tp);
    const uint32_t bytes = pairs * 16u;
    mbar_arrive_expect_tx(R.full + slot, uint32_t(R.narr) * bytes);
    float4* dst = const_cast<float4*>(R.slots) + size_t(slot) * R.slot_f4;
    const size_t arr_stride = size_t(P.pairB - P.pairA);    // pair arrays equally spaced in global memory
    for (int r = 0; r < R.narr; ++r) {
        const float4* src = P.pairA + size_t(r) * arr_stride + size_t(t) * R.tp;
        for (uint32_t o = 0; o < bytes; o += 32768u) {
            const uint32_t nb = bytes - o < 32768u ? bytes - o : 32768u;
            tma_bulk_g2s(reinterpret_cast<unsigned char*>(dst + size_t(r) * R.tp) + o,
                         reinterpret_cast<const unsigned char*>(src) + o, nb, R.full + slot);
        }
    }
}
// the warp is done with the tile in its current slot; the last warp to say so refills the slot
__device__ __forceinline__ void ring_release(const RolloutX2Params& P, SphSrc& S) {
    __syncwarp();
    if ((threadIdx.x & 31) == 0) {
        __threadfence_block();                              // this warp's reads of the slot are done
        const int old = atomicAdd(S.ring.done + S.pos.slot, 1);
        if (old == S.ring.consumers - 1) {
            S.ring.done[S.pos.slot] = 0;                    // nobody touches it before the refill has landed
            if (S.pos.v + kRingStages < S.ring.total) {
                int t = S.pos.t + kRingStages;
                while (t >= S.ring.nt) t -= S.ring.nt;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy reads before the async-proxy write
                ring_issue(P, S.ring, t, S.pos.slot);
            }
        }
    }
    S.pos.advance(S.ring.nt);
}

// visit (and release) the tiles of one pass without computing: a warp whose agent block has fewer chunks than the others
__device__ __forceinline__ void ring_skip_pass(const RolloutX2Params& P, SphSrc& S) {
    for (int t = 0; t < S.ring.nt; ++t) {
        mbar_wait(S.ring.full + S.pos.slot, S.pos.parity);
        ring_release(P, S);
    }
}

// One pass over the whole sphere set for this lane.  RING: tile by tile out of the ring, refinement as predicted by the
// caller (`hot`); otherwise the resident arrays with the two-pass refinement (sweep_any updates `hot`).
template <bool RING, int NA, bool FORCE, bool CULL, bool APF, bool MV, class RD>
__device__ __forceinline__ void sweep_src(const RolloutX2Params& P, SphSrc& S, int trips, int lane, int L, int logL, float tk,
                                          const float (&p)[NA][3], const float (&v)[NA][3], const RD& rd, float eps, unsigned mask,
                                          float thr, bool& hot, X2Acc<NA>& acc) {
    if (!RING) { sweep_any<NA, FORCE, CULL, APF, MV>(S.tA, S.tB, trips, lane, L, tk, p, v, rd, eps, mask, thr, hot, acc); return; }
    for (int t = 0; t < S.ring.nt; ++t) {
        mbar_wait(S.ring.full + S.pos.slot, S.pos.parity);
        const float4* tA = S.ring.slots + size_t(S.pos.slot) * S.ring.slot_f4;
        const float4* tB = tA + S.ring.tp;
        const int tt = (t == S.ring.nt - 1 ? S.ring.last_pairs : S.ring.tp) >> logL;
        if (FORCE && !hot) sweep_pass<NA, FORCE, CULL, APF, MV, false>(tA, tB, tt, lane, L, tk, p, v, rd, eps, mask, acc);
        else               sweep_pass<NA, FORCE, CULL, APF, MV, true>(tA, tB, tt, lane, L, tk, p, v, rd, eps, mask, acc);
        ring_release(P, S);
    }
}

// ring mode: does this warp have to refine the NEXT sweep?  dmin: the lane's clearance minima of the sweep just done,
// v: the agents' new velocities
template <int NA>
__device__ __forceinline__ bool ring_predict_hot(const float (&dmin)[NA], const float (&v)[NA][3], float dt, float thr, float umax_dt) {
    bool near = false;
#pragma unroll
    for (int a = 0; a < NA; ++a) near = near || (dmin[a] < thr + fmaf(dt, norm3f(v[a][0], v[a][1], v[a][2]), umax_dt));
    return __any_sync(0xffffffffu, near);
}

// Transposed butterfly over a full warp.  In: per-lane partial (x,y,z) of NA agents.  Out: every lane of
// half h (lanes 16h..16h+15; NA == 1: both halves) holds the warp total (X,Y,Z) of agent h.
template <int NA>
__device__ __forceinline__ void warp_sum3(const float (&x)[NA], const float (&y)[NA], const float (&z)[NA],
                                          int lane, float& X, float& Y, float& Z) {
    const unsigned full = 0xffffffffu;
    float u;
    (void)u;
    if (NA == 2) {
        const bool h16 = lane & 16;
        // step 16: lower half keeps agent 0, upper half keeps agent 1
        float kx = h16 ? x[NA - 1] : x[0], ky = h16 ? y[NA - 1] : y[0], kz = h16 ? z[NA - 1] : z[0];
        float sx = h16 ? x[0] : x[NA - 1], sy = h16 ? y[0] : y[NA - 1], sz = h16 ? z[0] : z[NA - 1];
        kx += __shfl_xor_sync(full, sx, 16); ky += __shfl_xor_sync(full, sy, 16); kz += __shfl_xor_sync(full, sz, 16);
        half_sum3(kx, ky, kz, lane, X, Y, Z);
    } else {
        const bool h16 = lane & 16, h8 = lane & 8;
        float kx = x[0], ky = y[0], kz = z[0];
        float r1 = __shfl_xor_sync(full, h16 ? kx : kz, 16);
        float r2 = __shfl_xor_sync(full, ky, 16);
        if (h16) kz += r1; else { kx += r1; ky += r2; }
        float send = h16 ? kz : (h8 ? kx : ky);
        float keep = h16 ? kz : (h8 ? ky : kx);
        u = keep + __shfl_xor_sync(full, send, 8);
        u += __shfl_xor_sync(full, u, 4);
        u += __shfl_xor_sync(full, u, 2);
        u += __shfl_xor_sync(full, u, 1);
        X = __shfl_sync(full, u, 0); Y = __shfl_sync(full, u, 8); Z = __shfl_sync(full, u, 16);
    }
}

// Plain xor butterfly for sub-warp groups (L < 32): every lane of the group gets every agent's totals.
template <int NA>
__device__ __forceinline__ void subwarp_allreduce(float (&x)[NA], float (&y)[NA], float (&z)[NA], float (&m)[NA],
                                                  int L, unsigned mask) {
    for (int off = L >> 1; off > 0; off >>= 1) {
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            x[a] += __shfl_xor_sync(mask, x[a], off);
            y[a] += __shfl_xor_sync(mask, y[a], off);
            z[a] += __shfl_xor_sync(mask, z[a], off);
            m[a] = fminf(m[a], __shfl_xor_sync(mask, m[a], off));
        }
    }
}

// One agent's per-step state update and cost accumulation (Eq. 6-11, 17-20), executed by the lane(s) that own it.
struct AgentX2 {
    float p[3], v[3], ap[3];
    int gid;                  // index of this agent in the caller's arrays
    float rd, kf;             // its detection radius and gain (uniform unless gmapp_set_agent_params was called)
    CostAcc ca;
    __device__ __forceinline__ void init(const RolloutX2Params& P, int i) {
        gid = agent_gid(P, i);
        rd = agent_rd(P, gid);
        kf = P.kf_arr ? P.kf_arr[gid] : P.k_circ;
        const float* s = P.agents_in + 6 * size_t(gid);
#pragma unroll
        for (int c = 0; c < 3; ++c) { p[c] = s[c]; v[c] = s[3 + c]; ap[c] = 0.0f; }
        ca.init(norm3f(P.goal[0] - p[0], P.goal[1] - p[1], P.goal[2] - p[2]));
    }
    __device__ __forceinline__ float rcg(const RolloutX2Params& P) const { return P.rcg_is_rd ? rd : P.rcg; }
    __device__ __forceinline__ float rco(const RolloutX2Params& P) const { return P.rco_is_rd ? rd : P.rco; }
    // Part of the state update that does not need the sphere sums (runs while the sums are still in flight):
    // e = goal - p, 1/|v| (MUFU.RSQ + Newton), |v|, and the attractor f_a = k_att e - k_damp v (Eq. 7).
    float ex, ey, ez, inv, nv, fax, fay, faz;
    __device__ __forceinline__ void pre(const RolloutX2Params& P) {
        ex = P.goal[0] - p[0]; ey = P.goal[1] - p[1]; ez = P.goal[2] - p[2];
        const float n2 = fmaf(v[0], v[0], fmaf(v[1], v[1], fmaf(v[2], v[2], kTiny)));
        inv = rsqrt_approx(n2);
        inv = inv * fmaf(-0.5f * n2 * inv, inv, 1.5f);
        nv = n2 * inv;
        fax = fmaf(P.k_att, ex, -P.k_damp * v[0]); fay = fmaf(P.k_att, ey, -P.k_damp * v[1]); faz = fmaf(P.k_att, ez, -P.k_damp * v[2]);
    }
    // The critical path once the sums B are known: f_r = k_f [((B.v)/|v|) v - |v| B] (BAC-CAB form of Eq. 2-3),
    // f = f_a + f_r (Eq. 6), v += vel_factor dt inv_mass f (Eq. 9-10), p += dt v (Eq. 11).
    template <bool APF>
    __device__ __forceinline__ void post(const RolloutX2Params& P, float bx, float by, float bz, float& fx, float& fy, float& fz) {
        if (APF) {                                         // Eq. 1: the sums are the force itself
            fx = fmaf(kf, bx, fax); fy = fmaf(kf, by, fay); fz = fmaf(kf, bz, faz);
        } else {
            const float A = fmaf(bx, v[0], fmaf(by, v[1], bz * v[2]));
            const float c1 = kf * inv * A, c2 = -kf * nv;
            fx = fmaf(c1, v[0], fmaf(c2, bx, fax)); fy = fmaf(c1, v[1], fmaf(c2, by, fay)); fz = fmaf(c1, v[2], fmaf(c2, bz, faz));
        }
        v[0] = fmaf(P.c_lin, fx, v[0]); v[1] = fmaf(P.c_lin, fy, v[1]); v[2] = fmaf(P.c_lin, fz, v[2]);
        p[0] = fmaf(P.dt, v[0], p[0]); p[1] = fmaf(P.dt, v[1], p[1]); p[2] = fmaf(P.dt, v[2], p[2]);
    }
    // costs of the pose the step started from (uses e = goal - p_old and that pose's clearance) and of the move
    __device__ __forceinline__ void costs(const RolloutX2Params& P, int k, float dmin, float fx, float fy, float fz) {
        ca.pose(norm3f(ex, ey, ez), dmin, rcg(P), rco(P));
        if (k >= 2) {                                                   // third difference = vf dt^2 (a_k - a_{k-1})
            float jx = fx - ap[0], jy = fy - ap[1], jz = fz - ap[2];
            ca.add_jerk(fmaf(jx, jx, fmaf(jy, jy, jz * jz)));
        }
        ap[0] = fx; ap[1] = fy; ap[2] = fz;
        ca.add_len(norm3f(v[0], v[1], v[2]));                           // |p_new - p| = dt |v_new|
    }
    // closed-loop re-planning: the state after snap_step steps (call right after post of step k)
    __device__ __forceinline__ void snapshot(const RolloutX2Params& P, int k) const {
        if (P.snap_out && k + 1 == P.snap_step) {
            float* o = P.snap_out + 6 * size_t(gid);
#pragma unroll
            for (int c = 0; c < 3; ++c) { o[c] = p[c]; o[3 + c] = v[c]; }
        }
        if (P.traj_out) {                                   // explored paths: every pose of every agent
            float* o = P.traj_out + 6 * (size_t(gid) * (P.steps + 1) + k + 1);
#pragma unroll
            for (int c = 0; c < 3; ++c) { o[c] = p[c]; o[3 + c] = v[c]; }
        }
    }
    __device__ __forceinline__ void finish(const RolloutX2Params& P, float dmin_final) {
        const int i = gid;
        ca.pose(norm3f(P.goal[0] - p[0], P.goal[1] - p[1], P.goal[2] - p[2]), dmin_final, rcg(P), rco(P));
        const float cj = P.vel_factor * P.dt * P.dt * P.inv_mass;
        const float Nk = float(P.steps) + 1.0f;
        const float Lp = P.dt * ca.sumV, J = cj * cj * ca.sumJ, d1 = ca.d1;
        float Cg = ca.sumG / Nk, Co = ca.sumO / Nk, Cp;
        if (Lp == 0.0f && d1 == 0.0f) Cp = 0.0f;
        else if (Lp >= d1) Cp = 1.0f - d1 / Lp;
        else Cp = 1.0f - Lp / d1;
        const float dt2 = P.dt * P.dt;
        const float Cs = fminf(1.0f, J / (Nk * dt2 * dt2 * P.a_max * P.a_max));
        float* out5 = P.cost + 5 * size_t(i);
        out5[0] = P.w_goal * Cg + P.w_obs * Co + P.w_path * Cp + P.w_smooth * Cs;
        out5[1] = Cg; out5[2] = Co; out5[3] = Cp; out5[4] = Cs;
        P.minclr[i] = ca.minclr;
        P.collided[i] = ca.collided;
        if (P.agents_out) {
            float* o = P.agents_out + 6 * size_t(i);
#pragma unroll
            for (int c = 0; c < 3; ++c) { o[c] = p[c]; o[3 + c] = v[c]; }
        }
    }
};

// ---------------------------------------------------------------------------------------------
// warp-level combine shared by the L >= 32 bodies: per-lane partials -> (X, Y, Z, D) of the agent owned by
// this lane's half (NA == 2: lanes 0-15 agent 0, lanes 16-31 agent 1; NA == 1: the one agent on all lanes)
// ---------------------------------------------------------------------------------------------
template <int NA, bool SC>
__device__ __forceinline__ void warp_combine(const X2Acc<NA>& acc, int lane, float& X, float& Y, float& Z, float& D) {
    float x[NA], y[NA], z[NA], dm[NA];
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        x[a] = acc_fold<SC>(acc.bx[a]); y[a] = acc_fold<SC>(acc.by[a]); z[a] = acc_fold<SC>(acc.bz[a]);
        dm[a] = fkey_inv(__reduce_min_sync(0xffffffffu, fkey(acc.dmin[a])));
    }
    warp_sum3<NA>(x, y, z, lane, X, Y, Z);
    D = (NA == 2 && (lane & 16)) ? dm[NA - 1] : dm[0];
}

// ---------------------------------------------------------------------------------------------
// epilogue side of the hand-over: add the W per-warp partials (x, y, z summed, w = min).  W is a power of two
// between 2 and 16; every case issues all its loads before the first add and adds as a tree, so the epilogue
// warp (the critical path of the latency-bound shapes) waits for one shared-memory round trip, not W.
// ---------------------------------------------------------------------------------------------
template <int WC>
__device__ __forceinline__ float4 sum_partials_n(const float4* q, int stride) {
    float4 t[WC];
#pragma unroll
    for (int w = 0; w < WC; ++w) t[w] = q[w * stride];
#pragma unroll
    for (int s = 1; s < WC; s <<= 1)
#pragma unroll
        for (int w = 0; w + s < WC; w += 2 * s) {
            t[w].x += t[w + s].x; t[w].y += t[w + s].y; t[w].z += t[w + s].z; t[w].w = fminf(t[w].w, t[w + s].w);
        }
    return t[0];
}
// NW = 2, 4, 8: exactly that many; NW = 0: n = 16 or 32 in chunks of eight
template <int NW>
__device__ __forceinline__ float4 sum_partials(const float4* q, int n, int stride) {
    if (NW > 0) return sum_partials_n<(NW > 0 ? NW : 2)>(q, stride);
    float4 t = sum_partials_n<8>(q, stride);
    for (int m = 8; m < n; m += 8) {
        const float4 o = sum_partials_n<8>(q + m * stride, stride);
        t.x += o.x; t.y += o.y; t.z += o.z; t.w = fminf(t.w, o.w);
    }
    return t;
}

// Group reduction done by the epilogue warp (multi-warp groups).  The sweep lanes leave their per-lane partials
// (x, y, z, dmin) in shared memory as part[NA][L]; lane l of the epilogue warp first adds L/32 of them (NA == 2:
// lanes 0-15 add L/16 of agent 0, lanes 16-31 of agent 1), then the warp finishes with a butterfly.
// One butterfly per group and step instead of one per sweep warp.  NW = partials per lane (L/32, NA == 2: L/16) when
// that is 2, 4 or 8, else 0: a template parameter so that the step loop of the epilogue warp has no dispatch in it.
template <int NA, int NW>
__device__ __forceinline__ float4 group_reduce(const float4* part, int L, int lane) {
    const unsigned full = 0xffffffffu;
    float4 t;
    if (NA == 2) t = sum_partials<NW>(part + (lane >> 4) * L + (lane & 15), L >> 4, 16);
    else         t = sum_partials<NW>(part + lane, L >> 5, 32);
    // plain xor butterfly on the four values (over the 16-lane half for two agents): the epilogue warp is the
    // critical path of the latency-bound shapes, and this form needs no hand-round of the sums at the end
    // (the transposed butterfly of the sweep-side reductions saves shuffles, which matters there, not here)
#pragma unroll
    for (int off = (NA == 2 ? 8 : 16); off > 0; off >>= 1) {
        t.x += __shfl_xor_sync(full, t.x, off);
        t.y += __shfl_xor_sync(full, t.y, off);
        t.z += __shfl_xor_sync(full, t.z, off);
        t.w = fminf(t.w, __shfl_xor_sync(full, t.w, off));
    }
    return t;
}

// ---------------------------------------------------------------------------------------------
// group body, L == 32: one warp per group does everything; agent a on lanes 0-15, agent b on lanes 16-31
// ---------------------------------------------------------------------------------------------
template <bool RING, int NA, bool CULL, bool APF, bool PER, bool XT, bool MV, bool ONE>
__device__ __forceinline__ void group_rollout_warp_n(const RolloutX2Params& P, SphSrc& S, int first_agent, int lane) {
    const int trips = ONE ? 1 : (S.n2p >> 5);              // ONE: at most 32 sphere pairs, straight-line sweep
    const int half = (NA == 2) ? (lane >> 4) : 0;
    const unsigned full = 0xffffffffu;
    AgentX2 me;
    me.init(P, first_agent + half);
    float p[NA][3], v[NA][3];
    RdSel<NA, PER> rd; rd.u = P.r_d;
    rd.v[0] = __shfl_sync(full, me.rd, 0);
    if (NA == 2) rd.v[NA - 1] = __shfl_sync(full, me.rd, 16);
    X2Acc<NA> acc;
    const float thr = lane_near_thr<APF>(RING ? P.pairB : S.tB, trips, lane, 32);
    bool hot = RING;                                       // ring mode: step 0 refines, later steps as predicted
    for (int k = 0; k <= P.steps; ++k) {
        const bool last = (k == P.steps);                  // pose S+1: distance-only pass
        const float tk = fmaf(float(k), P.dt, P.t0);       // obstacle time (moving spheres)
        if (NA == 2) {
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                p[0][i] = __shfl_sync(full, me.p[i], 0);       v[0][i] = __shfl_sync(full, me.v[i], 0);
                p[NA - 1][i] = __shfl_sync(full, me.p[i], 16); v[NA - 1][i] = __shfl_sync(full, me.v[i], 16);
            }
        } else {
#pragma unroll
            for (int i = 0; i < 3; ++i) { p[0][i] = me.p[i]; v[0][i] = me.v[i]; }
        }
        acc.clear();
        if (!last) sweep_src<RING, NA, true, CULL, APF, MV>(P, S, trips, lane, 32, 5, tk, p, v, rd, P.eps, full, thr, hot, acc);
        else       sweep_src<RING, NA, false, false, false, MV>(P, S, trips, lane, 32, 5, tk, p, v, rd, P.eps, full, thr, hot, acc);
        float X, Y, Z, D;
        warp_combine<NA, acc_scaled<APF, MV>()>(acc, lane, X, Y, Z, D);
        if (last) {
            if ((lane & 15) == 0 && (NA == 2 || lane == 0)) me.finish(P, D);
            return;
        }
        float fx, fy, fz;
        me.pre(P);
        me.template post<(APF || MV)>(P, X, Y, Z, fx, fy, fz);
        me.costs(P, k, D, fx, fy, fz);
        if (RING) {                                        // every lane needs both agents' new velocities
            float vn[NA][3];
#pragma unroll
            for (int i = 0; i < 3; ++i) { vn[0][i] = __shfl_sync(full, me.v[i], 0); if (NA == 2) vn[NA - 1][i] = __shfl_sync(full, me.v[i], 16); }
            hot = ring_predict_hot<NA>(acc.dmin, vn, P.dt, thr, S.umax_dt);
        }
        if ((lane & 15) == 0 && (NA == 2 || lane == 0)) { if (XT) me.snapshot(P, k); }
    }
}

template <bool RING, int NA, bool CULL, bool APF, bool PER, bool XT, bool MV>
__device__ __forceinline__ void group_rollout_warp(const RolloutX2Params& P, SphSrc& S, int first_agent, int lane) {
    if (!RING && S.n2p == 32) group_rollout_warp_n<false, NA, CULL, APF, PER, XT, MV, true>(P, S, first_agent, lane);
    else group_rollout_warp_n<RING, NA, CULL, APF, PER, XT, MV, false>(P, S, first_agent, lane);
}

// ---------------------------------------------------------------------------------------------
// many agents per CTA (more than two per warp): every warp owns a contiguous block of the CTA's agents and
// walks it in chunks of two inside each step; the persistent per-agent state (24 words) lives in a
// warp-private shared-memory record between visits.  No cross-warp traffic, no barriers, all warps busy.
// ---------------------------------------------------------------------------------------------
constexpr int kAgentRecWords = 24;      // p3 v3 ap3 | sumG cG sumO cO sumV cV sumJ cJ minclr d1 collided | gid rd kf | pad
__device__ __forceinline__ void agent_store(const AgentX2& a, float* r) {
    r[0] = a.p[0]; r[1] = a.p[1]; r[2] = a.p[2]; r[3] = a.v[0]; r[4] = a.v[1]; r[5] = a.v[2];
    r[6] = a.ap[0]; r[7] = a.ap[1]; r[8] = a.ap[2];
    r[9] = a.ca.sumG; r[10] = a.ca.cG; r[11] = a.ca.sumO; r[12] = a.ca.cO; r[13] = a.ca.sumV; r[14] = a.ca.cV;
    r[15] = a.ca.sumJ; r[16] = a.ca.cJ; r[17] = a.ca.minclr; r[18] = a.ca.d1; r[19] = __int_as_float(a.ca.collided);
    r[20] = __int_as_float(a.gid); r[21] = a.rd; r[22] = a.kf;
}
__device__ __forceinline__ void agent_load(AgentX2& a, const float* r) {
    a.p[0] = r[0]; a.p[1] = r[1]; a.p[2] = r[2]; a.v[0] = r[3]; a.v[1] = r[4]; a.v[2] = r[5];
    a.ap[0] = r[6]; a.ap[1] = r[7]; a.ap[2] = r[8];
    a.ca.sumG = r[9]; a.ca.cG = r[10]; a.ca.sumO = r[11]; a.ca.cO = r[12]; a.ca.sumV = r[13]; a.ca.cV = r[14];
    a.ca.sumJ = r[15]; a.ca.cJ = r[16]; a.ca.minclr = r[17]; a.ca.d1 = r[18]; a.ca.collided = __float_as_int(r[19]);
    a.gid = __float_as_int(r[20]); a.rd = r[21]; a.kf = r[22];
}

template <bool RING, int NA, bool CULL, bool APF, bool PER, bool XT, bool MV>
__device__ __forceinline__ void chunk_step(const RolloutX2Params& P, SphSrc& S, int agent0,
                                           int lane, int k, float thr, bool& hot, float* rec0) {
    const int n2p = S.n2p;
    const int half = (NA == 2) ? (lane >> 4) : 0;
    const unsigned full = 0xffffffffu;
    float* rec = rec0 + half * kAgentRecWords;
    AgentX2 me;
    agent_load(me, rec);
    float p[NA][3], v[NA][3];
    RdSel<NA, PER> rd; rd.u = P.r_d;
    if (NA == 2) {
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            p[0][i] = __shfl_sync(full, me.p[i], 0);       v[0][i] = __shfl_sync(full, me.v[i], 0);
            p[NA - 1][i] = __shfl_sync(full, me.p[i], 16); v[NA - 1][i] = __shfl_sync(full, me.v[i], 16);
        }
        rd.v[0] = __shfl_sync(full, me.rd, 0); rd.v[NA - 1] = __shfl_sync(full, me.rd, 16);
    } else {
#pragma unroll
        for (int i = 0; i < 3; ++i) { p[0][i] = me.p[i]; v[0][i] = me.v[i]; }
        rd.v[0] = me.rd;
    }
    const bool last = (k == P.steps);
    const float tk = fmaf(float(k), P.dt, P.t0);
    X2Acc<NA> acc;
    acc.clear();
    if (!last) sweep_src<RING, NA, true, CULL, APF, MV>(P, S, n2p >> 5, lane, 32, 5, tk, p, v, rd, P.eps, full, thr, hot, acc);
    else       sweep_src<RING, NA, false, false, false, MV>(P, S, n2p >> 5, lane, 32, 5, tk, p, v, rd, P.eps, full, thr, hot, acc);
    float X, Y, Z, D;
    warp_combine<NA, acc_scaled<APF, MV>()>(acc, lane, X, Y, Z, D);
    const bool writer = (lane & 15) == 0 && (NA == 2 || lane == 0);
    if (last) {
        if (writer) me.finish(P, D);
        return;
    }
    float fx, fy, fz;
    me.pre(P);
    me.template post<(APF || MV)>(P, X, Y, Z, fx, fy, fz);
    me.costs(P, k, D, fx, fy, fz);
    if (RING) {
        float vn[NA][3];
#pragma unroll
        for (int i = 0; i < 3; ++i) { vn[0][i] = __shfl_sync(full, me.v[i], 0); if (NA == 2) vn[NA - 1][i] = __shfl_sync(full, me.v[i], 16); }
        hot = ring_predict_hot<NA>(acc.dmin, vn, P.dt, thr, S.umax_dt);
    }
    if (writer) { if (XT) me.snapshot(P, k); }
    __syncwarp();                                         // every lane has read the record before it is rewritten
    if (writer) agent_store(me, rec);
    __syncwarp();
}

template <bool RING, bool CULL, bool APF, bool PER, bool XT, bool MV>
__device__ __forceinline__ void warp_rollout_chunks(const RolloutX2Params& P, SphSrc& S, int first_agent, int n_mine, int rounds,
                                                    int lane, float* recs) {
    // records of this warp's agents: recs[i * kAgentRecWords], i < n_mine
    for (int i = lane; i < n_mine; i += 32) {
        AgentX2 a;
        a.init(P, first_agent + i);
        agent_store(a, recs + i * kAgentRecWords);
    }
    __syncwarp();
    const float thr = lane_near_thr<APF>(RING ? P.pairB : S.tB, S.n2p >> 5, lane, 32);
    // refined-mode flag of each chunk (chunks beyond 64 share bits: conservative in ring mode -- a shared bit is the OR
    // of its chunks there -- and harmless otherwise); ring mode starts refined
    u64 hotbits = RING ? ~0ull : 0ull;
    for (int k = 0; k <= P.steps; ++k) {
        u64 next = 0ull;
        for (int i = 0; i < n_mine; i += 2) {
            const int c = (i >> 1) & 63;
            bool hot = (hotbits >> c) & 1ull;
            if (i + 2 <= n_mine) chunk_step<RING, 2, CULL, APF, PER, XT, MV>(P, S, first_agent + i, lane, k, thr, hot, recs + i * kAgentRecWords);
            else                 chunk_step<RING, 1, CULL, APF, PER, XT, MV>(P, S, first_agent + i, lane, k, thr, hot, recs + i * kAgentRecWords);
            if (RING) next |= u64(hot) << c;
            else hotbits = (hotbits & ~(1ull << c)) | (u64(hot) << c);
        }
        if (RING) {
            hotbits = next;
            for (int r = (n_mine + 1) >> 1; r < rounds; ++r) ring_skip_pass(P, S);     // keep the CTA's tile sequence
        }
    }
}

// ---------------------------------------------------------------------------------------------
// group bodies, L >= 64: W = L/32 sweep warps + ONE epilogue warp per group.
// shared exchange area per group: part[NA][L] float4 (per-lane x, y, z, dmin), state[2][NA][2] float4 (p,0), (v,0).
// One arrive/sync pair per direction and step is race-free: the epilogue warp has consumed part (its loads feed the
// state it publishes) before it arrives at bar_state, and the sweep warps write part again only after that barrier;
// state is double-buffered by step parity.
//   sweep warp k:    write part -> arrive(bar_part) -> sync(bar_state) -> read state[k&1]
//   epilogue warp k: sync(bar_part) -> reduce part -> integrate -> write state[k&1] -> arrive(bar_state) -> costs
// ---------------------------------------------------------------------------------------------
template <bool RING, int NA, bool CULL, bool APF, bool PER, bool MV, bool ONE, int LC = 0>
__device__ __forceinline__ void group_sweep_warps_n(const RolloutX2Params& P, SphSrc& S,
                                                    int first_agent, int lane_in_group, int group_in_cta, float4* xch,
                                                    int gL = 0, int glogL = 0) {
    // LC > 0: the width as a compile-time constant (the unrolled trips then address the tile with immediate offsets);
    // gL > 0: the group's own width (mixed widths in one CTA); else the launch's uniform P.L
    const int L = LC ? LC : (gL ? gL : P.L), logL = LC ? (LC == 128 ? 7 : 6) : (gL ? glogL : P.logL);
    const int n2p = S.n2p;
    // n2p is a multiple of L: the same trip count on every lane.  ONE: a single trip (as many lanes as sphere pairs,
    // the latency-bound shapes): known at compile time, so the sweep is straight-line code without loop control
    const int trips = ONE ? 1 : (n2p >> logL);
    const unsigned full = 0xffffffffu;
    float4* part = xch;                                    // [NA][L]
    const float4* state = xch + 2 * L;                   // [2][NA][2]
    const int bar_part = 1 + 2 * group_in_cta, bar_state = 2 + 2 * group_in_cta, nbar = L + 32;
    float p[NA][3], v[NA][3];
    RdSel<NA, PER> rd; rd.u = P.r_d;
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        const int gid = agent_gid(P, first_agent + a);
        const float* s = P.agents_in + 6 * size_t(gid);
        rd.v[a] = agent_rd(P, gid);
#pragma unroll
        for (int i = 0; i < 3; ++i) { p[a][i] = s[i]; v[a][i] = s[3 + i]; }
    }
    X2Acc<NA> acc;
    const float thr = lane_near_thr<APF>(RING ? P.pairB : S.tB, trips, lane_in_group, L);
    bool hot = RING;
    for (int k = 0; k <= P.steps; ++k) {
        const bool last = (k == P.steps);
        const float tk = fmaf(float(k), P.dt, P.t0);
        acc.clear();
        if (!last) sweep_src<RING, NA, true, CULL, APF, MV>(P, S, trips, lane_in_group, L, logL, tk, p, v, rd, P.eps, full, thr, hot, acc);
        else       sweep_src<RING, NA, false, false, false, MV>(P, S, trips, lane_in_group, L, logL, tk, p, v, rd, P.eps, full, thr, hot, acc);
#pragma unroll
        for (int a = 0; a < NA; ++a) {                     // per-lane partials; the epilogue warp reduces them
            constexpr bool SC = acc_scaled<APF, MV>();
            part[a * L + lane_in_group] = make_float4(acc_fold<SC>(acc.bx[a]), acc_fold<SC>(acc.by[a]), acc_fold<SC>(acc.bz[a]), acc.dmin[a]);
        }
        const int par = k & 1;
        named_bar_arrive(bar_part, nbar);
        if (last) return;
        named_bar_sync(bar_state, nbar);
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            const float4 sp = state[(par * NA + a) * 2], sv = state[(par * NA + a) * 2 + 1];
            p[a][0] = sp.x; p[a][1] = sp.y; p[a][2] = sp.z; v[a][0] = sv.x; v[a][1] = sv.y; v[a][2] = sv.z;
        }
        if (RING) hot = ring_predict_hot<NA>(acc.dmin, v, P.dt, thr, S.umax_dt);
    }
}

template <bool RING, int NA, bool CULL, bool APF, bool PER, bool MV, int LC = 0>
__device__ __forceinline__ void group_sweep_warps(const RolloutX2Params& P, SphSrc& S,
                                                  int first_agent, int lane_in_group, int group_in_cta, float4* xch,
                                                  int gL = 0, int glogL = 0) {
    if (GMAPP_X2_L128 && LC > 0 && !RING) {                 // mixed-width mode: the group's width is known at compile time
        group_sweep_warps_n<false, NA, CULL, APF, PER, MV, false, LC>(P, S, first_agent, lane_in_group, group_in_cta, xch);
        return;
    }
    if (!RING && (S.n2p >> (gL ? glogL : P.logL)) == 1) group_sweep_warps_n<false, NA, CULL, APF, PER, MV, true>(P, S, first_agent, lane_in_group, group_in_cta, xch, gL, glogL);
    else if (GMAPP_X2_L128 && !RING && !gL && P.L == 128) group_sweep_warps_n<false, NA, CULL, APF, PER, MV, false, 128>(P, S, first_agent, lane_in_group, group_in_cta, xch);
    else group_sweep_warps_n<RING, NA, CULL, APF, PER, MV, false>(P, S, first_agent, lane_in_group, group_in_cta, xch, gL, glogL);
}

template <int NA, bool APF, bool XT, int NW>   // APF here = "the sums are the force itself" (APF heuristic or moving spheres)
__device__ __forceinline__ void group_epilogue_warp_n(const RolloutX2Params& P, int first_agent, int lane,
                                                    int group_in_cta, float4* xch) {
    const int half = (NA == 2) ? (lane >> 4) : 0;
    const float4* part = xch;
    float4* state = xch + 2 * P.L;
    const int bar_part = 1 + 2 * group_in_cta, bar_state = 2 + 2 * group_in_cta, nbar = P.L + 32;
    AgentX2 me;
    me.init(P, first_agent + half);
    for (int k = 0; k <= P.steps; ++k) {
        const bool last = (k == P.steps);
        const int par = k & 1;
        me.pre(P);                                         // everything that does not need the sphere sums
        named_bar_sync(bar_part, nbar);
        const float4 t = group_reduce<NA, NW>(part, P.L, lane);
        if (last) {
            if ((lane & 15) == 0 && (NA == 2 || lane == 0)) me.finish(P, t.w);
            return;
        }
        float fx, fy, fz;
        me.template post<APF>(P, t.x, t.y, t.z, fx, fy, fz);
        if ((lane & 15) == 0 && (NA == 2 || lane == 0)) {
            state[(par * NA + half) * 2] = make_float4(me.p[0], me.p[1], me.p[2], 0.0f);
            state[(par * NA + half) * 2 + 1] = make_float4(me.v[0], me.v[1], me.v[2], 0.0f);
        }
        named_bar_arrive(bar_state, nbar);
        me.costs(P, k, t.w, fx, fy, fz);                   // off the critical path: the sweep warps are already running
        if ((lane & 15) == 0 && (NA == 2 || lane == 0)) { if (XT) me.snapshot(P, k); }
    }
}

template <int NA, bool APF, bool XT>
__device__ __forceinline__ void group_epilogue_warp(const RolloutX2Params& P, int first_agent, int lane,
                                                    int group_in_cta, float4* xch) {
    const int n = P.L >> (NA == 2 ? 4 : 5);                // partials per epilogue lane
    if (n == 4) group_epilogue_warp_n<NA, APF, XT, 4>(P, first_agent, lane, group_in_cta, xch);
    else if (n == 8) group_epilogue_warp_n<NA, APF, XT, 8>(P, first_agent, lane, group_in_cta, xch);
    else if (n == 2) group_epilogue_warp_n<NA, APF, XT, 2>(P, first_agent, lane, group_in_cta, xch);
    else group_epilogue_warp_n<NA, APF, XT, 0>(P, first_agent, lane, group_in_cta, xch);
}

// ---------------------------------------------------------------------------------------------
// 5 to 7 groups per CTA (9 to 14 agents): MIXED GROUP WIDTHS and one epilogue warp serving TWO groups.
// With G groups of two sweep warps each the four schedulers of the SM carry unequal numbers of sweep warps (2048 agents: 14
// warps, 4 : 4 : 3 : 3) and an epilogue warp per group makes 21 warps, which cuts the register budget from 96 to 80.  Instead
// the CTA always has 16 sweep warps: the first y = 2 G - 8 groups are 2 warps wide (L = 64), the other 8 - G groups 4 warps
// (L = 128).  y is even and the 2-wide groups come first, so every run of four consecutive warps holds two 2-wide groups or
// one 4-wide group and every scheduler carries the same number of agent-sweeps per step; a one-agent group (odd agent
// count) is the last group and therefore 4 wide.  ceil(G / 2) shared epilogue warps: 19 or 20 warps, 96 registers.  An
// epilogue warp serves its groups in a fixed order each step; the second group's hand-over waits for the first one's
// (~0.3 us against a sweep of several us).
// NA1 = 0: the warp's second group does not exist (odd group count, or the CTA's agents end before it).
// ---------------------------------------------------------------------------------------------
template <int NA>
struct EpiSide {
    AgentX2 me;
    const float4* part; float4* state;
    int bar_part, bar_state, half, L;
    __device__ __forceinline__ void init(const RolloutX2Params& P, int first_agent, int lane, int group_in_cta, float4* xch, int L_) {
        half = (NA == 2) ? (lane >> 4) : 0;
        L = L_;                                             // this group's width: 64 or 128 lanes
        part = xch; state = xch + 2 * L;
        bar_part = 1 + 2 * group_in_cta; bar_state = 2 + 2 * group_in_cta;
        me.init(P, first_agent + half);
    }
    // one step of this group: returns false after the final pose
    template <bool APF, bool XT>
    __device__ __forceinline__ void step(const RolloutX2Params& P, int k, int lane, float& dmin, float& fx, float& fy, float& fz) {
        const bool last = (k == P.steps);
        const int par = k & 1, nbar = L + 32;
        const bool writer = (lane & 15) == 0 && (NA == 2 || lane == 0);
        me.pre(P);
        named_bar_sync(bar_part, nbar);
        // partials per epilogue lane: L / 16 (two agents) or L / 32; the group is 2 or 4 sweep warps wide (a uniform branch)
        float4 t;
        if (L == 64) t = group_reduce<NA, (NA == 2 ? 4 : 2)>(part, 64, lane);
        else         t = group_reduce<NA, (NA == 2 ? 8 : 4)>(part, 128, lane);
        dmin = t.w;
        if (last) { if (writer) me.finish(P, t.w); return; }
        me.template post<APF>(P, t.x, t.y, t.z, fx, fy, fz);
        if (writer) {
            state[(par * NA + half) * 2] = make_float4(me.p[0], me.p[1], me.p[2], 0.0f);
            state[(par * NA + half) * 2 + 1] = make_float4(me.v[0], me.v[1], me.v[2], 0.0f);
        }
        named_bar_arrive(bar_state, nbar);
    }
};

template <int NA0, int NA1, bool APF, bool XT>
__device__ __forceinline__ void group_epilogue_warp2_n(const RolloutX2Params& P, int first0, int first1, int lane, int g0,
                                                       float4* xch0, float4* xch1, int L0, int L1) {
    EpiSide<NA0> s0;
    EpiSide<(NA1 > 0 ? NA1 : 1)> s1;
    s0.init(P, first0, lane, g0, xch0, L0);
    if (NA1 > 0) s1.init(P, first1, lane, g0 + 1, xch1, L1);
    for (int k = 0; k <= P.steps; ++k) {
        float d0, d1 = 0.0f, f0x, f0y, f0z, f1x, f1y, f1z;
        s0.template step<APF, XT>(P, k, lane, d0, f0x, f0y, f0z);
        if (NA1 > 0) s1.template step<APF, XT>(P, k, lane, d1, f1x, f1y, f1z);
        if (k == P.steps) return;
        s0.me.costs(P, k, d0, f0x, f0y, f0z);              // off the critical path: both groups' sweep warps are running
        if ((lane & 15) == 0 && (NA0 == 2 || lane == 0)) { if (XT) s0.me.snapshot(P, k); }
        if (NA1 > 0) {
            s1.me.costs(P, k, d1, f1x, f1y, f1z);
            if ((lane & 15) == 0 && (NA1 == 2 || lane == 0)) { if (XT) s1.me.snapshot(P, k); }
        }
    }
}

// na0, na1: agents of the warp's two groups (na0 in {1, 2}; na1 in {0, 1, 2}, and na1 > 0 only if na0 == 2)
template <bool APF, bool XT>
__device__ __forceinline__ void group_epilogue_warp2(const RolloutX2Params& P, int first0, int na0, int na1, int lane, int g0,
                                                     float4* xch0, float4* xch1, int L0, int L1) {
    const int first1 = first0 + 2;
    if (na0 >= 2 && na1 >= 2) group_epilogue_warp2_n<2, 2, APF, XT>(P, first0, first1, lane, g0, xch0, xch1, L0, L1);
    else if (na0 >= 2 && na1 == 1) group_epilogue_warp2_n<2, 1, APF, XT>(P, first0, first1, lane, g0, xch0, xch1, L0, L1);
    else if (na0 >= 2) group_epilogue_warp2_n<2, 0, APF, XT>(P, first0, first1, lane, g0, xch0, xch1, L0, L1);
    else group_epilogue_warp2_n<1, 0, APF, XT>(P, first0, first1, lane, g0, xch0, xch1, L0, L1);
}

// ---------------------------------------------------------------------------------------------
// group body, L < 32 (several groups per warp): plain butterfly, every lane integrates its group's agents
// ---------------------------------------------------------------------------------------------
template <int NA, bool CULL, bool APF, bool PER, bool XT, bool MV>
__device__ __forceinline__ void group_rollout_narrow(const RolloutX2Params& P, const SphSrc& S,
                                                     int first_agent, int lane_in_group) {
    const float4* tA = S.tA; const float4* tB = S.tB; const int n2p = S.n2p;
    const unsigned mask = __activemask();
    const int trips = n2p >> P.logL;                       // n2p is a multiple of L
    AgentX2 ag[NA];
    float p[NA][3], v[NA][3];
    RdSel<NA, PER> rd; rd.u = P.r_d;
#pragma unroll
    for (int a = 0; a < NA; ++a) { ag[a].init(P, first_agent + a); rd.v[a] = ag[a].rd; }
    X2Acc<NA> acc;
    const float thr = lane_near_thr<APF>(tB, trips, lane_in_group, P.L);
    bool hot = false;
    for (int k = 0; k <= P.steps; ++k) {
        const bool last = (k == P.steps);
        const float tk = fmaf(float(k), P.dt, P.t0);
#pragma unroll
        for (int a = 0; a < NA; ++a)
#pragma unroll
            for (int i = 0; i < 3; ++i) { p[a][i] = ag[a].p[i]; v[a][i] = ag[a].v[i]; }
        acc.clear();
        if (!last) sweep_any<NA, true, CULL, APF, MV>(tA, tB, trips, lane_in_group, P.L, tk, p, v, rd, P.eps, mask, thr, hot, acc);
        else       sweep_any<NA, false, false, false, MV>(tA, tB, trips, lane_in_group, P.L, tk, p, v, rd, P.eps, mask, thr, hot, acc);
        float x[NA], y[NA], z[NA], dm[NA];
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            constexpr bool SC = acc_scaled<APF, MV>();
            x[a] = acc_fold<SC>(acc.bx[a]); y[a] = acc_fold<SC>(acc.by[a]); z[a] = acc_fold<SC>(acc.bz[a]);
            dm[a] = acc.dmin[a];
        }
        subwarp_allreduce<NA>(x, y, z, dm, P.L, mask);
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            if (last) { if (lane_in_group == 0) ag[a].finish(P, dm[a]); continue; }
            float fx, fy, fz;
            ag[a].pre(P);
            ag[a].template post<(APF || MV)>(P, x[a], y[a], z[a], fx, fy, fz);
            ag[a].costs(P, k, dm[a], fx, fy, fz);
            if (lane_in_group == 0) { if (XT) ag[a].snapshot(P, k); }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// the kernel: one launch per planning cycle
// ---------------------------------------------------------------------------------------------
// AT = agents per group (1 or 2); MODE 0: L < 32 (sub-warp groups), 1: L == 32 (one warp per group),
// 2: L >= 64 (W sweep warps + one epilogue warp per group; threads [0, G L) sweep, [G L, G L + 32 G) epilogue);
// 4: many agents per CTA, each warp walks its block of agents in chunks of two (state records in shared memory);
// STAGE 1 = sphere pairs staged in shared memory by TMA bulk copies (a template parameter on purpose: as a run-time
// choice the tile pointers become generic and every LDS turns into a generic LD, measured 10 % slower)
// XT = extras: the state snapshot of gmapp_replan and the trajectory output (kept out of the plain kernels: the few
// extra stores in the epilogue perturb the register allocation of the sweep warps by 3 %)
template <int AT, int MODE, bool CULL, int STAGE, int MAXT, bool APF, bool XT, bool MV>
__global__ void __launch_bounds__(MAXT == 576 ? 640 : MAXT, 1) k_rollout_x2(const __grid_constant__ RolloutX2Params P) {   // (MAXT 576 = tag of the mixed-width variant: 19 or 20 warps)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw);
    constexpr bool RING = (STAGE == 2);
    constexpr int NARR = MV ? 4 : 2;                        // pair arrays A, B (, U, V), equally spaced in global memory
    SphSrc S;
    S.tA = P.pairA; S.tB = P.pairB;
    const int tid = threadIdx.x;
    int n2p = P.n2p;
    if (P.count_dev) {                                      // built sphere world: the count never went to the host
        const int n = min(*P.count_dev, P.n_cap), h = (n + 1) >> 1;
        n2p = min(P.n2p, ((h + P.L - 1) >> P.logL) << P.logL);
    }
    S.n2p = n2p;
    const int cta_first = blockIdx.x * P.agents_per_cta;
    int cta_end = cta_first + P.agents_per_cta;
    if (cta_end > P.n_agents) cta_end = P.n_agents;
    const int n_cta = cta_end - cta_first;
    int rounds = 1;                                         // ring passes per step (mode 4: agent chunks per warp)
    if (STAGE == 1) {
        float4* tile = reinterpret_cast<float4*>(smem_raw + P.tile_off);
        if (tid == 0) { mbar_init(bar, 1); fence_mbar_init(); }
        __syncthreads();
        if (tid == 0 && n2p > 0) {
            const uint32_t bytes = uint32_t(n2p) * 16u;
            mbar_arrive_expect_tx(bar, NARR * bytes);
            const uint32_t chunk = 32768u;
            for (int r = 0; r < NARR; ++r) {
                const unsigned char* src = reinterpret_cast<const unsigned char*>(P.pairA + size_t(r) * (P.pairB - P.pairA));
                for (uint32_t o = 0; o < bytes; o += chunk) {
                    const uint32_t nb = bytes - o < chunk ? bytes - o : chunk;
                    tma_bulk_g2s(reinterpret_cast<unsigned char*>(tile) + r * bytes + o, src + o, nb, bar);
                }
            }
        }
        S.tA = tile;
        S.tB = tile + n2p;
    }
    if (RING) {
        // consumer warps of this CTA (warps that return at once because they have no agent do not count)
        const int n_sweep_threads = int(blockDim.x);
        int consumers;
        if (MODE == 2 && AT == 2 && MAXT == 576) {          // mixed group widths: the sweep warps of the groups that have agents
            const int G = (P.agents_per_cta + 1) / 2, y = 2 * G - 8, ga = (n_cta + 1) / 2;
            consumers = 0;
            for (int g = 0; g < G && g < ga; ++g) consumers += g < y ? 2 : 4;
        } else if (MODE == 2) {
            const int G = (P.agents_per_cta + AT - 1) / AT, ga = (n_cta + AT - 1) / AT;
            consumers = (ga < G ? ga : G) * (P.L >> 5);
        } else if (MODE == 4) {
            const int nw = n_sweep_threads >> 5;
            consumers = n_cta < nw ? n_cta : nw;
            const int most = (n_cta + nw - 1) / nw;          // largest agent block of a warp
            rounds = (most + 1) >> 1;
        } else {
            const int G = n_sweep_threads >> 5;
            consumers = n_cta < G ? n_cta : G;
        }
        S.ring.full = reinterpret_cast<uint64_t*>(smem_raw + P.ring_off);
        S.ring.done = reinterpret_cast<int*>(S.ring.full + kRingStages);
        S.ring.slots = reinterpret_cast<const float4*>(smem_raw + P.tile_off);
        S.ring.tp = P.ring_tp; S.ring.slot_f4 = NARR * P.ring_tp; S.ring.narr = NARR;
        S.ring.nt = (n2p + P.ring_tp - 1) / P.ring_tp;
        S.ring.last_pairs = n2p - (S.ring.nt - 1) * P.ring_tp;
        S.ring.consumers = consumers; S.ring.total = (P.steps + 1) * rounds * S.ring.nt;
        S.pos.slot = 0; S.pos.parity = 0u; S.pos.t = 0; S.pos.v = 0;
        S.umax_dt = MV ? P.sph_stats[1] * P.dt : 0.0f;
        if (tid == 0) {
            for (int i = 0; i < kRingStages; ++i) { mbar_init(S.ring.full + i, 1); S.ring.done[i] = 0; }
            fence_mbar_init();
            // the first kRingStages visits; after that the last warp to release a slot refills it
            for (int i = 0, t = 0; i < kRingStages && i < S.ring.total; ++i) { ring_issue(P, S.ring, t, i); if (++t == S.ring.nt) t = 0; }
        }
        __syncthreads();
    } else {
        S.ring.full = nullptr; S.ring.done = nullptr; S.ring.slots = nullptr;
        S.ring.tp = S.ring.slot_f4 = S.ring.nt = S.ring.last_pairs = S.ring.narr = S.ring.consumers = S.ring.total = 0;
        S.pos.slot = 0; S.pos.parity = 0u; S.pos.t = S.pos.v = 0; S.umax_dt = 0.0f;
    }
    constexpr int NA2 = (AT == 2) ? 2 : 1;
    if (MODE == 2 && AT == 2 && MAXT == 576) {
        // mixed group widths (see group_epilogue_warp2): 16 sweep warps, groups [0, y) 2 warps wide, [y, G) 4 warps wide
        const int G = (P.agents_per_cta + 1) / 2, y = 2 * G - 8, w = tid >> 5;
        const bool is_epi = w >= 16;
        float4* xbase = reinterpret_cast<float4*>(smem_raw + P.xch_off);
        // group g: lanes, first sweep warp, exchange area (2 L + 8 float4 per group)
        #define GMAPP_MIX_L(g) ((g) < y ? 64 : 128)
        #define GMAPP_MIX_W0(g) ((g) < y ? 2 * (g) : 2 * y + 4 * ((g) - y))
        #define GMAPP_MIX_X(g) (xbase + ((g) < y ? (g) * 136 : y * 136 + ((g) - y) * 264))
        if (is_epi) {
            const int g0 = 2 * (w - 16), first = cta_first + 2 * g0, na = cta_end - first;
            if (g0 >= G || na <= 0) return;
            int na1 = (g0 + 1 < G) ? na - 2 : 0;
            if (na1 > 2) na1 = 2;
            if (na1 < 0) na1 = 0;
            group_epilogue_warp2<(APF || MV), XT>(P, first, na, na1, tid & 31, g0, GMAPP_MIX_X(g0), GMAPP_MIX_X(g0 + 1),
                                                  GMAPP_MIX_L(g0), GMAPP_MIX_L(g0 + 1));
            select_tail<GMAPP_FUSED_SELECT_X2 != 0>(P.sel, P.cost, P.collided, (na >= 2 ? 2 : 1) + na1, tid & 31);
            return;
        }
        const int g = w < 2 * y ? (w >> 1) : y + ((w - 2 * y) >> 2);
        const int first = cta_first + 2 * g, na = cta_end - first;
        if (STAGE == 1 && n2p > 0) mbar_wait(bar, 0);
        if (g >= G || na <= 0) return;
        const int gL = GMAPP_MIX_L(g), glogL = g < y ? 6 : 7, lane_in_group = tid - 32 * GMAPP_MIX_W0(g);
        float4* xch = GMAPP_MIX_X(g);
        // Compile-time widths (64 / 128) for the two-agent groups -- unless this CTA also has a one-agent group next to 128-wide
        // two-agent groups: three different sweep bodies running on one SM measured 10 % slower than two (1500 agents, 11 per
        // CTA: 1.146 -> 1.270 ms), so such a CTA keeps the run-time width for all its groups.  (The per-agent-radius variant and
        // the one-agent group always use the run-time width: fewer instantiations.)
        const int ga = (n_cta + 1) >> 1;
        const bool lc_ok = !((n_cta & 1) && ga - 1 > y);
        if (na >= 2) {
            if (P.rd_arr || !lc_ok) { if (P.rd_arr) group_sweep_warps<RING, 2, CULL, APF, true, MV>(P, S, first, lane_in_group, g, xch, gL, glogL); else group_sweep_warps<RING, 2, CULL, APF, false, MV>(P, S, first, lane_in_group, g, xch, gL, glogL); }
            else if (g < y) group_sweep_warps<RING, 2, CULL, APF, false, MV, 64>(P, S, first, lane_in_group, g, xch, gL, glogL);
            else group_sweep_warps<RING, 2, CULL, APF, false, MV, 128>(P, S, first, lane_in_group, g, xch, gL, glogL);
        }
        else { if (P.rd_arr) group_sweep_warps<RING, 1, CULL, APF, true, MV>(P, S, first, lane_in_group, g, xch, gL, glogL); else group_sweep_warps<RING, 1, CULL, APF, false, MV>(P, S, first, lane_in_group, g, xch, gL, glogL); }
        return;
        #undef GMAPP_MIX_L
        #undef GMAPP_MIX_W0
        #undef GMAPP_MIX_X
    }
    if (MODE == 2) {
        const int G = (P.agents_per_cta + AT - 1) / AT;
        const int n_sweep = G * P.L;
        const bool is_epi = tid >= n_sweep;
        const int group_in_cta = is_epi ? ((tid - n_sweep) >> 5) : (tid >> P.logL);
        const int first = cta_first + group_in_cta * AT;
        const int na = cta_end - first;
        float4* xch = reinterpret_cast<float4*>(smem_raw + P.xch_off) + group_in_cta * (2 * P.L + 8);
        if (is_epi) {                                      // the epilogue warps never touch the sphere tile
            if (na <= 0) return;
            if (AT == 2 && na >= 2) group_epilogue_warp<NA2, (APF || MV), XT>(P, first, tid & 31, group_in_cta, xch);
            else group_epilogue_warp<1, (APF || MV), XT>(P, first, tid & 31, group_in_cta, xch);
            select_tail<GMAPP_FUSED_SELECT_X2 != 0>(P.sel, P.cost, P.collided, (AT == 2 && na >= 2) ? 2 : 1, tid & 31);    // S8: the last warp selects
            return;
        }
        if (STAGE == 1 && n2p > 0) mbar_wait(bar, 0);
        if (na <= 0) return;
        const int lane_in_group = tid & (P.L - 1);
        if (AT == 2 && na >= 2) { if (P.rd_arr) group_sweep_warps<RING, NA2, CULL, APF, true, MV>(P, S, first, lane_in_group, group_in_cta, xch); else group_sweep_warps<RING, NA2, CULL, APF, false, MV>(P, S, first, lane_in_group, group_in_cta, xch); }
        else { if (P.rd_arr) group_sweep_warps<RING, 1, CULL, APF, true, MV>(P, S, first, lane_in_group, group_in_cta, xch); else group_sweep_warps<RING, 1, CULL, APF, false, MV>(P, S, first, lane_in_group, group_in_cta, xch); }
        return;
    }
    if (MODE == 4) {
        // balanced contiguous split of the CTA's agents over its warps
        const int nw = int(blockDim.x) >> 5, w = tid >> 5;
        const int base = n_cta / nw, rem = n_cta % nw;
        const int start = w * base + (w < rem ? w : rem), n_mine = base + (w < rem ? 1 : 0);
        if (STAGE == 1 && n2p > 0) mbar_wait(bar, 0);
        if (n_mine <= 0) return;
        float* recs = reinterpret_cast<float*>(smem_raw + P.rec_off) + start * kAgentRecWords;
        { if (P.rd_arr) warp_rollout_chunks<RING, CULL, APF, true, XT, MV>(P, S, cta_first + start, n_mine, rounds, tid & 31, recs); else warp_rollout_chunks<RING, CULL, APF, false, XT, MV>(P, S, cta_first + start, n_mine, rounds, tid & 31, recs); }
        select_tail<GMAPP_FUSED_SELECT_X2 != 0>(P.sel, P.cost, P.collided, n_mine, tid & 31);
        return;
    }
    const int group_in_cta = tid >> P.logL;
    const int lane_in_group = tid & (P.L - 1);
    int first = cta_first + group_in_cta * AT;
    int na = cta_end - first;
    if (MODE == 1 && AT == 2) {
        // one warp per group, G warps for n <= 2 G agents: the first n - G groups take two agents, the others one, so that
        // a warp count that is a multiple of 4 loads the four schedulers equally (28 agents on 16 warps = 12 x 2 + 4 x 1,
        // 7 agent-sweeps per scheduler; 14 warps x 2 would put 8 on two schedulers and 6 on the others)
        const int G = int(blockDim.x) >> 5, n = n_cta;
        const int g2 = n - G < 0 ? 0 : (n - G > G ? G : n - G);
        first = cta_first + (group_in_cta < g2 ? 2 * group_in_cta : g2 + group_in_cta);
        na = group_in_cta < g2 ? 2 : (first < cta_end ? 1 : 0);
    }
    if (STAGE == 1 && n2p > 0) mbar_wait(bar, 0);
    if (na <= 0) return;
    if (MODE == 1) {
        if (AT == 2 && na >= 2) { if (P.rd_arr) group_rollout_warp<RING, NA2, CULL, APF, true, XT, MV>(P, S, first, lane_in_group); else group_rollout_warp<RING, NA2, CULL, APF, false, XT, MV>(P, S, first, lane_in_group); }
        else { if (P.rd_arr) group_rollout_warp<RING, 1, CULL, APF, true, XT, MV>(P, S, first, lane_in_group); else group_rollout_warp<RING, 1, CULL, APF, false, XT, MV>(P, S, first, lane_in_group); }
        select_tail<GMAPP_FUSED_SELECT_X2 != 0>(P.sel, P.cost, P.collided, (AT == 2 && na >= 2) ? 2 : 1, tid & 31);
    } else {
        if (AT == 2 && na >= 2) { if (P.rd_arr) group_rollout_narrow<NA2, CULL, APF, true, XT, MV>(P, S, first, lane_in_group); else group_rollout_narrow<NA2, CULL, APF, false, XT, MV>(P, S, first, lane_in_group); }
        else { if (P.rd_arr) group_rollout_narrow<1, CULL, APF, true, XT, MV>(P, S, first, lane_in_group); else group_rollout_narrow<1, CULL, APF, false, XT, MV>(P, S, first, lane_in_group); }
        if (lane_in_group == 0) select_tail_serial<GMAPP_FUSED_SELECT_X2 != 0>(P.sel, P.cost, P.collided, (AT == 2 && na >= 2) ? 2 : 1);   // sub-warp groups
    }
}

#ifdef GMAPP_MAIN_TU
// pack (xyz, r) [+ velocities] -> sphere-pair arrays A, B (, U, V), `stride` float4 apart; R = r + r_agent stored
// negated; sentinel pairs (far away, at rest) up to n2_fill
__global__ void k_pack_pairs(const float4* __restrict__ sph_raw, const float4* __restrict__ svel, int n, int n2_fill,
                             float r_agent, float4* __restrict__ pairs, int stride) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n2_fill) return;
    const float far = kFar;
    float4 s0 = make_float4(far, far, far, 0.0f), s1 = s0, u0 = make_float4(0, 0, 0, 0), u1 = u0;
    if (2 * j < n) { s0 = sph_raw[2 * j]; s0.w += r_agent; if (svel) u0 = svel[2 * j]; }
    if (2 * j + 1 < n) { s1 = sph_raw[2 * j + 1]; s1.w += r_agent; if (svel) u1 = svel[2 * j + 1]; }
    pairs[j] = make_float4(s0.x, s1.x, s0.y, s1.y);
    pairs[stride + j] = make_float4(s0.z, s1.z, -s0.w, -s1.w);
    if (svel) {
        pairs[2 * stride + j] = make_float4(u0.x, u1.x, u0.y, u1.y);
        pairs[3 * stride + j] = make_float4(u0.z, u1.z, 0.0f, 0.0f);
    }
}

#endif  // GMAPP_MAIN_TU

}  // namespace gmapp
