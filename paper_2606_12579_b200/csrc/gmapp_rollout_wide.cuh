// gmapp_rollout_wide.cuh -- rollout kernel for 6D motor agents (static or moving spheres) when a group of lanes spans
// several warps (L >= 64, <= 4 groups per CTA: the few-agents / many-spheres shape of config 4).
//
// Same machine mapping as the multi-warp mode of gmapp_rollout_x2.cuh: W = L/32 sweep warps per group evaluate the
// pair sums (packed f32x2 pair math; per-pair relative velocity for moving spheres), combine
// them inside the warp (transposed butterfly + REDUX.MIN) and post them to shared memory; ONE epilogue warp per
// group adds the W partials, updates the agent(s) and publishes (p, world velocity) for the next sweep.  The 6D
// update is split so that everything that does not need the sphere sums -- the SE(3) log map of Eq. 8, the
// torque, the rotor increment exp(dt w), the new rotor -- runs BEFORE the epilogue warp waits for the sums; after
// the wait only R^T f_r, the new twist, the translation of exp(dt v) and two rotations remain (Eq. 9-11).
// In the scalar kernel the whole 6D update ran redundantly on every lane of the group and took 60 % of the time.
//
// Shares nothing with oracle/.
#pragma once
#include "gmapp_rollout_x2.cuh"

namespace gmapp {


// ---------------------------------------------------------------------------------------------
// epilogue-side agent models.  Interface: init, pre (no sums needed), post (sums known -> new state, pub[6] =
// position and WORLD linear velocity for the sweep warps), costs, finish.
// ---------------------------------------------------------------------------------------------
// DIRECT: the sums are the force itself (moving spheres or APF); else the BAC-CAB assembly of Eq. 2-3
template <bool DIRECT>
struct EpiPose6 {
    Pose6 x;
    Quat rg; Vec3 pg;
    float pub[6];
    // computed by pre(): old position, torque-updated angular velocity, new rotor, exp coefficients, force without f_r
    Vec3 pos, w_new, phi, fpre, td, dp, dp1, dp2;
    Quat r_new;
    float Bc, Cc;
    int gid; float rd, kf;
    CostAcc ca;
    __device__ __forceinline__ float rcg(const RolloutParams& P) const { return P.rcg_is_rd ? rd : P.rcg; }
    __device__ __forceinline__ float rco(const RolloutParams& P) const { return P.rco_is_rd ? rd : P.rco; }
    __device__ __forceinline__ void init(const RolloutParams& P, int i) {
        gid = agent_gid(P, i); rd = agent_rd(P, gid); kf = agent_kf(P, gid);
        x = load_pose6(P.agents_in + 14 * size_t(gid));
        rg = Quat{P.goal[0], P.goal[1], P.goal[2], P.goal[3]};
        Quat dg = Quat{P.goal[4], P.goal[5], P.goal[6], P.goal[7]};
        motor_normalise(rg, dg);
        pg = motor_translation(rg, dg);
        ca.init(norm3f(pg.x - x.p.x, pg.y - x.p.y, pg.z - x.p.z));
        dp1 = v3(0, 0, 0); dp2 = v3(0, 0, 0);
        const Vec3 pdot = qrot(x.r, x.nu);
        pub[0] = x.p.x; pub[1] = x.p.y; pub[2] = x.p.z; pub[3] = pdot.x; pub[4] = pdot.y; pub[5] = pdot.z;
    }
    // Eq. 8 log map, torque, w update, rotation part of exp(dt v), new rotor: none of it needs the sphere sums
    __device__ __forceinline__ void pre(const RolloutParams& P) {
        pos = x.p;
        const Quat qrel = qmul(qconj(x.r), rg);
        const Vec3 trel = qrot_inv(x.r, pg - pos);
        Vec3 ew, ev;
        se3_log_from_quat(qrel, trel, ew, ev);
        const Vec3 tau = fma3(P.k_att_rot, ew, (-P.k_damp_rot) * x.w);
        fpre = fma3(P.k_att, ev, (-P.k_damp) * x.nu);
        w_new = fma3(P.c_rot, tau, x.w);                                   // Eq. 9-10, rotational block
        phi = P.dt * w_new;
        float ch, sh_over_th;
        se3_exp_coeffs(phi, ch, sh_over_th, Bc, Cc);
        const Quat rd = Quat{ch, sh_over_th * phi.x, sh_over_th * phi.y, sh_over_th * phi.z};
        r_new = qmul(x.r, rd);                                             // Eq. 11, rotor part of M <- M exp(dt v)
        Quat dz = Quat{0, 0, 0, 0};
        motor_normalise(r_new, dz);
    }
    __device__ __forceinline__ void post(const RolloutParams& P, float bx, float by, float bz) {
        Vec3 fr;
        if (DIRECT) fr = kf * v3(bx, by, bz);
        else cf_force_static(kf, bx, by, bz, pub[3], pub[4], pub[5], fr.x, fr.y, fr.z);
        const Vec3 f = fpre + qrot_inv(x.r, fr);                           // Eq. 6 in the body frame (reading G18)
        x.nu = fma3(P.c_lin, f, x.nu);                                     // Eq. 9-10, linear block
        const Vec3 rho = P.dt * x.nu;
        const Vec3 wr = cross(phi, rho);
        const Vec3 wwr = cross(phi, wr);
        td = fma3(Cc, wwr, fma3(Bc, wr, rho));                             // translation of exp(dt v)
        dp = qrot(x.r, td);                                                // world displacement p_new - p
        x.p = x.p + dp;
        x.r = r_new;
        x.w = w_new;
        const Vec3 pdot = qrot(x.r, x.nu);                                 // world linear velocity for the next sweep
        pub[0] = x.p.x; pub[1] = x.p.y; pub[2] = x.p.z; pub[3] = pdot.x; pub[4] = pdot.y; pub[5] = pdot.z;
    }
    __device__ __forceinline__ void costs(const RolloutParams& P, int k, float dmin) {
        ca.pose(norm3f(pg.x - pos.x, pg.y - pos.y, pg.z - pos.z), dmin, rcg(P), rco(P));
        ca.add_len(norm3f(td.x, td.y, td.z));
        if (k >= 2) {
            const Vec3 t3 = dp - 2.0f * dp1 + dp2;                         // p4 - 3 p3 + 3 p2 - p1 from displacements
            ca.add_jerk(dot(t3, t3));
        }
        dp2 = dp1; dp1 = dp;
    }
    __device__ __forceinline__ void finish(const RolloutParams& P, float dmin) {
        const int i = gid;
        ca.pose(norm3f(pg.x - x.p.x, pg.y - x.p.y, pg.z - x.p.z), dmin, rcg(P), rco(P));
        ca.finish(P, ca.sumV, ca.sumJ, P.cost + 5 * size_t(i));
        P.minclr[i] = ca.minclr;
        P.collided[i] = ca.collided;
        if (P.agents_out) write_pose6(x, P.agents_out + 14 * size_t(i));
    }
    __device__ __forceinline__ void snapshot(const RolloutParams& P, int k) const {
        if (P.snap_out && k + 1 == P.snap_step) write_pose6(x, P.snap_out + 14 * size_t(gid));
        if (P.traj_out) write_pose6(x, P.traj_out + 14 * (size_t(gid) * (P.steps + 1) + k + 1));
    }
};

// ---------------------------------------------------------------------------------------------
// group bodies (protocol and hazard argument as in gmapp_rollout_x2.cuh, multi-warp mode)
// exchange area per group: part[NA][L] float4 (per-lane partials, reduced by the epilogue warp), state[2][NA][2] float4
// ---------------------------------------------------------------------------------------------
// sweep warps: packed f32x2 sweeps over sphere pairs; tile = A, B (, U, V when MOVING) arrays of n2p float4 each
template <int NA, bool MOVING, bool CULL, bool APF, bool PER>
__device__ __forceinline__ void wide_sweep_warps(const RolloutParams& P, const float4* tile, int astride, int n2p, int first_agent,
                                                 int lane_in_group, int group_in_cta, float4* xch) {
    const unsigned full = 0xffffffffu;
    float4* part = xch;
    const float4* state = xch + NA * P.L;
    const int bar_part = 1 + 2 * group_in_cta, bar_state = 2 + 2 * group_in_cta, nbar = P.L + 32;
    const int trips = n2p >> P.logL;                       // n2p is a multiple of L
    const float4* tA = tile; const float4* tB = tile + astride;       // (U, V follow at the same spacing)
    float p[NA][3], v[NA][3];
    RdSel<NA, PER> rd; rd.u = P.r_d;
#pragma unroll
    for (int a = 0; a < NA; ++a) rd.v[a] = agent_rd(P, agent_gid(P, first_agent + a));
    // the start (p, world velocity) comes from the epilogue warp too (6D: needs the motor algebra): parity-1 buffer
    named_bar_sync(bar_state, nbar);
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        const float4 sp = state[(1 * NA + a) * 2], sv = state[(1 * NA + a) * 2 + 1];
        p[a][0] = sp.x; p[a][1] = sp.y; p[a][2] = sp.z; v[a][0] = sv.x; v[a][1] = sv.y; v[a][2] = sv.z;
    }
    X2Acc<NA> acc;
    const float thr = lane_near_thr<APF>(tB, trips, lane_in_group, P.L);     // two-pass distance refinement (gmapp_rollout_x2.cuh)
    bool hot = false;
    for (int k = 0; k <= P.steps; ++k) {
        const bool last = (k == P.steps);
        const float tk = fmaf(float(k), P.dt, P.t0);
        acc.clear();
        if (!last) sweep_any<NA, true, CULL, APF, MOVING>(tA, tB, trips, lane_in_group, P.L, tk, p, v, rd, P.eps, full, thr, hot, acc);
        else       sweep_any<NA, false, false, false, MOVING>(tA, tB, trips, lane_in_group, P.L, tk, p, v, rd, P.eps, full, thr, hot, acc);
#pragma unroll
        for (int a = 0; a < NA; ++a) {                     // per-lane partials; the epilogue warp reduces them
            constexpr bool SC = acc_scaled<APF, MOVING>();
            part[a * P.L + lane_in_group] = make_float4(acc_fold<SC>(acc.bx[a]), acc_fold<SC>(acc.by[a]), acc_fold<SC>(acc.bz[a]), acc.dmin[a]);
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
    }
}

template <class Model, int NA, int NW>
__device__ __forceinline__ void wide_epilogue_warp(const RolloutParams& P, int first_agent, int lane,
                                                   int group_in_cta, float4* xch) {
    const int half = (NA == 2) ? (lane >> 4) : 0;
    const bool writer = (lane & 15) == 0 && (NA == 2 || lane == 0);
    const float4* part = xch;
    float4* state = xch + NA * P.L;
    const int bar_part = 1 + 2 * group_in_cta, bar_state = 2 + 2 * group_in_cta, nbar = P.L + 32;
    Model me;
    me.init(P, first_agent + half);
    // hand the start state to the sweep warps through the parity-1 buffer (step 0 publishes into parity 0)
    if (writer) {
        state[(1 * NA + half) * 2] = make_float4(me.pub[0], me.pub[1], me.pub[2], 0.0f);
        state[(1 * NA + half) * 2 + 1] = make_float4(me.pub[3], me.pub[4], me.pub[5], 0.0f);
    }
    named_bar_arrive(bar_state, nbar);
    me.pre(P);
    for (int k = 0; k <= P.steps; ++k) {
        const bool last = (k == P.steps);
        const int par = k & 1;
        named_bar_sync(bar_part, nbar);
        const float4 t = group_reduce<NA, NW>(part, P.L, lane);
        if (last) {
            if (writer) me.finish(P, t.w);
            select_tail<GMAPP_FUSED_SELECT_WIDE != 0>(P.sel, P.cost, P.collided, NA, lane);
            return;
        }
        me.post(P, t.x, t.y, t.z);
        if (writer) {
            state[(par * NA + half) * 2] = make_float4(me.pub[0], me.pub[1], me.pub[2], 0.0f);
            state[(par * NA + half) * 2 + 1] = make_float4(me.pub[3], me.pub[4], me.pub[5], 0.0f);
        }
        named_bar_arrive(bar_state, nbar);
        // off the critical path of the sweep warps; the costs of this step and the sum-free part of the next
        // step sit in one block so their independent instruction chains interleave
        me.costs(P, k, t.w);
        if (writer) me.snapshot(P, k);
        me.pre(P);
    }
}

// ---------------------------------------------------------------------------------------------
// 6D agents, two epilogue warps per group.  With zero repulsive torque (reading G18) the rotational dynamics
// (r, w) never sees the sphere sums, so a ROT warp runs it on its own -- log of the relative rotation, torque, new
// angular velocity, rotor increment, new rotor -- one step ahead, and hands a 5 x float4 record per step to the LIN
// warp: [r_k] [e_w, c2] [phi, B] [r_{k+1}] [w_{k+1}, C].  The LIN warp does what needs the position and the sums.
// The single-warp epilogue spent ~520 dependent instructions per step on one warp and was the bottleneck of config 4;
// split, the chain per step is max(rot, lin).
// Hand-over by two named barriers per group, strictly alternating so that barrier generations never overlap:
//   rot step k:  compute record k -> sync(empty) [k >= 1: lin has read record k-1] -> write -> arrive(full)
//   lin step k:  sync(full) -> read record k -> arrive(empty) -> ... the usual epilogue step
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void wide_rot_warp(const RolloutParams& P, int agent, int lane, int group_in_cta, float4* rec) {
    const int bar_full = 9 + 2 * group_in_cta, bar_empty = 10 + 2 * group_in_cta;
    const int gid = agent_gid(P, agent);
    Pose6 x = load_pose6(P.agents_in + 14 * size_t(gid));
    Quat rg = Quat{P.goal[0], P.goal[1], P.goal[2], P.goal[3]}, dg = Quat{P.goal[4], P.goal[5], P.goal[6], P.goal[7]};
    motor_normalise(rg, dg);
    for (int k = 0; k < P.steps; ++k) {
        Vec3 ew; float c2;
        se3_log_rot(qmul(qconj(x.r), rg), ew, c2);
        const Vec3 tau = fma3(P.k_att_rot, ew, (-P.k_damp_rot) * x.w);
        const Vec3 w_new = fma3(P.c_rot, tau, x.w);                        // Eq. 9-10, rotational block
        const Vec3 phi = P.dt * w_new;
        float ch, sh_over_th, Bc, Cc;
        se3_exp_coeffs(phi, ch, sh_over_th, Bc, Cc);
        const Quat rd = Quat{ch, sh_over_th * phi.x, sh_over_th * phi.y, sh_over_th * phi.z};
        Quat r_new = qmul(x.r, rd);                                        // Eq. 11, rotor part
        Quat dz = Quat{0, 0, 0, 0};
        motor_normalise(r_new, dz);
        if (k >= 1) named_bar_sync(bar_empty, 64);
        if (lane == 0) {
            rec[0] = make_float4(x.r.w, x.r.x, x.r.y, x.r.z);
            rec[1] = make_float4(ew.x, ew.y, ew.z, c2);
            rec[2] = make_float4(phi.x, phi.y, phi.z, Bc);
            rec[3] = make_float4(r_new.w, r_new.x, r_new.y, r_new.z);
            rec[4] = make_float4(w_new.x, w_new.y, w_new.z, Cc);
        }
        named_bar_arrive(bar_full, 64);
        x.r = r_new; x.w = w_new;
    }
    if (P.steps >= 1) named_bar_sync(bar_empty, 64);                       // balance the lin warp's last arrive
}

template <bool DIRECT, int NW>
__device__ __forceinline__ void wide_lin_warp(const RolloutParams& P, int agent, int lane, int group_in_cta,
                                              float4* xch, const float4* rec) {
    const float4* part = xch;
    float4* state = xch + P.L;
    const int bar_part = 1 + 2 * group_in_cta, bar_state = 2 + 2 * group_in_cta, nbar = P.L + 32;
    const int bar_full = 9 + 2 * group_in_cta, bar_empty = 10 + 2 * group_in_cta;
    const bool writer = lane == 0;
    EpiPose6<DIRECT> me;
    me.init(P, agent);
    if (writer) {
        state[(1 * 1 + 0) * 2] = make_float4(me.pub[0], me.pub[1], me.pub[2], 0.0f);
        state[(1 * 1 + 0) * 2 + 1] = make_float4(me.pub[3], me.pub[4], me.pub[5], 0.0f);
    }
    named_bar_arrive(bar_state, nbar);
    Vec3 ew = v3(0, 0, 0); float c2 = 0.0f;
    for (int k = 0; k <= P.steps; ++k) {
        const bool last = (k == P.steps);
        const int par = k & 1;
        if (!last) {
            named_bar_sync(bar_full, 64);
            const float4 a0 = rec[0], a1 = rec[1], a2 = rec[2], a3 = rec[3], a4 = rec[4];
            named_bar_arrive(bar_empty, 64);
            me.x.r = Quat{a0.x, a0.y, a0.z, a0.w};
            ew = v3(a1.x, a1.y, a1.z); c2 = a1.w;
            me.phi = v3(a2.x, a2.y, a2.z); me.Bc = a2.w;
            me.r_new = Quat{a3.x, a3.y, a3.z, a3.w};
            me.w_new = v3(a4.x, a4.y, a4.z); me.Cc = a4.w;
            // the part of Eq. 8 / Eq. 7 that needs the position: e_v = V^-1(e_w) R^T (p_g - p), f without f_r
            me.pos = me.x.p;
            const Vec3 ev = se3_log_lin(ew, c2, qrot_inv(me.x.r, me.pg - me.pos));
            me.fpre = fma3(P.k_att, ev, (-P.k_damp) * me.x.nu);
        }
        named_bar_sync(bar_part, nbar);
        const float4 t = group_reduce<1, NW>(part, P.L, lane);
        if (last) {
            if (writer) me.finish(P, t.w);
            select_tail<GMAPP_FUSED_SELECT_WIDE != 0>(P.sel, P.cost, P.collided, 1, lane);
            return;
        }
        me.post(P, t.x, t.y, t.z);
        if (writer) {
            state[(par * 1 + 0) * 2] = make_float4(me.pub[0], me.pub[1], me.pub[2], 0.0f);
            state[(par * 1 + 0) * 2 + 1] = make_float4(me.pub[3], me.pub[4], me.pub[5], 0.0f);
        }
        named_bar_arrive(bar_state, nbar);
        me.costs(P, k, t.w);
        if (writer) me.snapshot(P, k);
    }
}

// ---------------------------------------------------------------------------------------------
// the kernel: threads [0, G L) sweep, [G L, G L + 32 G) one epilogue warp per group; G <= 4, L >= 64
// (or 64 G: a LIN and a ROT warp per group); one 6D motor agent per group
// ---------------------------------------------------------------------------------------------
template <bool MOVING, bool CULL, int STAGE, bool APF>
__global__ void __launch_bounds__(640, 1) k_rollout_wide(const __grid_constant__ RolloutParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw);
    const int tid = threadIdx.x;
    constexpr int NARR = MOVING ? 4 : 2;                    // pair arrays: A, B (, U, V)
    int n2p = P.n2p;
    if (P.count_dev) {                                      // built sphere world: sweep only the pairs holding real spheres
        const int n = min(*P.count_dev, P.n_cap), h = (n + 1) >> 1;
        n2p = min(P.n2p, ((h + P.L - 1) >> P.logL) << P.logL);
    }
    const float4* tile = P.pairA;                           // stage 0: read the pair arrays from global memory / L2
    int astride = P.pair_stride;
    if (STAGE == 1) {
        float4* t = reinterpret_cast<float4*>(smem_raw + P.tile_off);
        if (tid == 0) { mbar_init(bar, 1); fence_mbar_init(); }
        __syncthreads();
        if (tid == 0 && n2p > 0) {
            const uint32_t bytes = uint32_t(n2p) * 16u;
            mbar_arrive_expect_tx(bar, NARR * bytes);
            const uint32_t chunk = 32768u;
            for (int r = 0; r < NARR; ++r) {
                const unsigned char* src = reinterpret_cast<const unsigned char*>(P.pairA + size_t(r) * P.pair_stride);
                for (uint32_t o = 0; o < bytes; o += chunk) {
                    const uint32_t nb = bytes - o < chunk ? bytes - o : chunk;
                    tma_bulk_g2s(reinterpret_cast<unsigned char*>(t) + r * bytes + o, src + o, nb, bar);
                }
            }
        }
        tile = t;
        astride = n2p;
    }
    const int cta_first = blockIdx.x * P.agents_per_cta;
    int cta_end = cta_first + P.agents_per_cta;
    if (cta_end > P.n_agents) cta_end = P.n_agents;
    const int G = P.agents_per_cta;
    const int n_sweep = G * P.L;
    const bool is_epi = tid >= n_sweep;
    const int group_in_cta = is_epi ? ((tid - n_sweep) >> 5) : (tid >> P.logL);
    const int first = cta_first + group_in_cta;
    const int na = cta_end - first;
    float4* xch = reinterpret_cast<float4*>(smem_raw + P.red_off) + group_in_cta * (P.L + 8);
    if (P.two_warp_epi) {
        // threads [n_sweep, n_sweep + 32 G): lin warps; [n_sweep + 32 G, n_sweep + 64 G): rot warps
        if (tid >= n_sweep) {
            const int e = (tid - n_sweep) >> 5, g = e % G;
            const int ag = cta_first + g;
            if (ag >= cta_end) return;
            float4* base = reinterpret_cast<float4*>(smem_raw + P.red_off);
            float4* xg = base + g * (P.L + 8);
            float4* rec = base + G * (P.L + 8) + 5 * g;
            const int n = P.L >> 5;                        // partials per lane of the reducing warp (NW, 0 = 16)
            if (e >= G) wide_rot_warp(P, ag, tid & 31, g, rec);
            else if (n == 8) wide_lin_warp<(MOVING || APF), 8>(P, ag, tid & 31, g, xg, rec);
            else if (n == 4) wide_lin_warp<(MOVING || APF), 4>(P, ag, tid & 31, g, xg, rec);
            else if (n == 2) wide_lin_warp<(MOVING || APF), 2>(P, ag, tid & 31, g, xg, rec);
            else wide_lin_warp<(MOVING || APF), 0>(P, ag, tid & 31, g, xg, rec);
            return;
        }
    } else if (is_epi) {
        if (na <= 0) return;
        const int lane = tid & 31;
        if ((P.L >> 5) == 4) wide_epilogue_warp<EpiPose6<(MOVING || APF)>, 1, 4>(P, first, lane, group_in_cta, xch);   // 4 groups: L = 128
        else wide_epilogue_warp<EpiPose6<(MOVING || APF)>, 1, 2>(P, first, lane, group_in_cta, xch);                 //           or L = 64
        return;
    }
    if (STAGE == 1 && n2p > 0) mbar_wait(bar, 0);
    if (na <= 0) return;
    const int lane_in_group = tid & (P.L - 1);
    { if (P.rd_arr) wide_sweep_warps<1, MOVING, CULL, APF, true>(P, tile, astride, n2p, first, lane_in_group, group_in_cta, xch); else wide_sweep_warps<1, MOVING, CULL, APF, false>(P, tile, astride, n2p, first, lane_in_group, group_in_cta, xch); }
}

}  // namespace gmapp
