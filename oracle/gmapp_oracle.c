/*
 * gmapp_oracle.c  --  FP64 CPU oracle for the G-MAPP multi-agent vector-field rollout.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or helper with paper_2606_12579_b200/csrc (the CUDA path); the CUDA path never
 * calls it.  Plain C99, scalar loops, double precision, one agent after another; OpenMP over
 * agents is used ONLY when `threads > 1` is asked for (the timed CPU baseline), never for parity.
 *
 * It follows the paper step by step, in the paper's order and notation (PAPER.md = the text of
 * arxiv/paper_2606_12579).  No algebraic shortcut of the CUDA path appears here: the circular-field
 * force is the literal double cross product of Eq. 2-3, path length and jerk are literal position
 * differences (Eq. 19-20), the sphere sum is a plain sequential sum.  Where the paper is silent or
 * garbled the reading taken is the one listed in DESIGN.md ("Readings", G1..G34) and named here.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1 F.v = 0, P2 c.n = 0, P3 zero outside r_d,
 * P4 closed-form magnitude, P5 hand-computed single-sphere cases, P6 mirror / rotation / permutation
 * symmetry, P7 Galilean, P8 no-obstacle closed form (matrix power), P9 multi-step golden by hand,
 * P10 SE(3) exp/log vs scipy expm/logm and 6D == 3D reduction, P11 cost closed forms,
 * P12 agent independence, P13 brute-force numpy restatement, P14 APF (Eq. 1 under reading N1): hand-computed
 * single-sphere cases, F = -grad of the Khatib potential, superposition and mirror symmetry.
 * P16 (tests/test_oracle_pins_6d.py) the 6D rollout against T <- T expm(dt hat(twist)), e = vee(logm(T^-1 T_g)) on
 * 4x4 matrices with the closed-form force, random orientations + translation error + repulsion (fixes every
 * transpose / multiplication order of pose6_wrench and orc_rollout_pose6), P17 rigid-motion equivariance of the 6D
 * rollout, P18 quat_to_R hand cases + scipy, P19 the diagnostics scale / margins / kappa by hand from P5-A.
 * parity unpinned (fixed by DESIGN.md readings only, the paper gives no value to pin them to):
 * G16 (the 1/2 of Eq. 10 is taken as printed), G18 (frame of the 6D repulsion), G19 (N_k = S+1),
 * G23 (default constants), G24 (collision-first selection key).
 */
#include <math.h>
#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif
#include <stddef.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    double k_circ;                 /* k_f of Eq. 2; applied once (G31)           */
    double k_att, k_damp;          /* linear blocks of K, D in Eq. 7             */
    double k_att_rot, k_damp_rot;  /* rotational blocks of K, D (6D only)                       */
    double inv_mass, inv_inertia;  /* diagonal of the "inertia tensor" of Eq. 9 (G15)           */
    double vel_factor;             /* the printed 1/2 of Eq. 10 (G16)                           */
    double r_influence;            /* r_d                                                       */
    double r_agent;                /* r_a of Alg. 1                              */
    double eps_dist;               /* epsilon of Alg. 1 line 6                   */
    double w_goal, w_obs, w_path, w_smooth;   /* Eq. 16 weights                                 */
    double r_cost_goal, r_cost_obs;           /* Eq. 17/18 radii; 0 => r_influence (G20)        */
    double a_max;                  /* Eq. 20                                                    */
    int heuristic;                 /* 0 = circular field / MFI (Eq. 2-3); 1 = APF (Eq. 1)       */
} orc_gains;

/* ------------------------------------------------------------------ small vector helpers */
static double dot3(const double a[3], const double b[3]) { return a[0]*b[0] + a[1]*b[1] + a[2]*b[2]; }
static double norm3(const double a[3]) { return sqrt(dot3(a, a)); }
static void cross3(const double a[3], const double b[3], double o[3]) {
    o[0] = a[1]*b[2] - a[2]*b[1];
    o[1] = a[2]*b[0] - a[0]*b[2];
    o[2] = a[0]*b[1] - a[1]*b[0];
}
static void mat3_mul(const double A[9], const double B[9], double C[9]) {
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
        double s = 0.0;
        for (int k = 0; k < 3; ++k) s += A[3*i+k] * B[3*k+j];
        C[3*i+j] = s;
    }
}
static void mat3_vec(const double A[9], const double x[3], double y[3]) {
    for (int i = 0; i < 3; ++i) y[i] = A[3*i]*x[0] + A[3*i+1]*x[1] + A[3*i+2]*x[2];
}
static void mat3T_vec(const double A[9], const double x[3], double y[3]) {
    for (int i = 0; i < 3; ++i) y[i] = A[i]*x[0] + A[3+i]*x[1] + A[6+i]*x[2];
}
static void hat3(const double w[3], double W[9]) {
    W[0] = 0; W[1] = -w[2]; W[2] = w[1];
    W[3] = w[2]; W[4] = 0; W[5] = -w[0];
    W[6] = -w[1]; W[7] = w[0]; W[8] = 0;
}

/* ------------------------------------------------------------------ one agent-sphere pair
 * Alg. 1 lines 5-9 with Eq. 2-3 as CALC_HEURISTIC.
 *   d  = p_O - p_a                         (G1: centre minus agent)
 *   ds = ||d|| - (r_a + r_O)               (Alg. 1 line 6, G2)
 *   gate: ds <= r_d                        (Alg. 1 line 7, G9/G30)
 *   dO = max(ds, eps)                      (Alg. 1 line 6)
 *   ddot = v_agent - u_obstacle            (G5)
 *   c  = ddot - n (n . ddot), n = d/||d||  (Eq. 3, G4)
 *   B  = c x ddot                          (G3)
 *   f  = k_f/dO * (ddot/||ddot||) x B      (Eq. 2; k_f once, G31; ||ddot|| = 0 or ||d|| = 0 => 0, G7)
 * APF (heuristic 1, Eq. 1, reading N1 in DESIGN.md: Khatib form on the clamped
 * surface distance): f = k_f (1/dO - 1/r_d) / dO^2 * (p - p_O)/||p - p_O||.
 * Returns the gate decision; *ds_out always holds the unclamped surface distance. */
static int pair_force(const double p[3], const double v[3], const double c[3], double r,
                      const double u[3], const orc_gains* g, double f[3], double* ds_out)
{
    double d[3] = { c[0] - p[0], c[1] - p[1], c[2] - p[2] };
    double dist = norm3(d);
    double ds = dist - (g->r_agent + r);
    *ds_out = ds;
    f[0] = f[1] = f[2] = 0.0;
    if (!(ds <= g->r_influence)) return 0;
    double dO = fmax(ds, g->eps_dist);
    if (g->heuristic == 1) {
        if (dist > 0.0) {
            double m = g->k_circ * (1.0 / dO - 1.0 / g->r_influence) / (dO * dO);
            for (int i = 0; i < 3; ++i) f[i] = m * (-d[i] / dist);
        }
        return 1;
    }
    double vr[3] = { v[0] - u[0], v[1] - u[1], v[2] - u[2] };
    double nv = norm3(vr);
    if (nv > 0.0 && dist > 0.0) {
        double n[3] = { d[0] / dist, d[1] / dist, d[2] / dist };
        double ndv = dot3(n, vr);
        double cur[3] = { vr[0] - n[0]*ndv, vr[1] - n[1]*ndv, vr[2] - n[2]*ndv };   /* Eq. 3 */
        double B[3], vhat[3] = { vr[0] / nv, vr[1] / nv, vr[2] / nv }, F[3];
        cross3(cur, vr, B);                                                        /* B = c x ddot */
        cross3(vhat, B, F);                                                        /* Eq. 2 */
        double k = g->k_circ / dO;
        f[0] = k * F[0]; f[1] = k * F[1]; f[2] = k * F[2];
    }
    return 1;
}

/* exported for the single-pair pins (P1, P2, P4, P5, P7) */
int orc_pair_force(const double* p, const double* v, const double* c, double r, const double* u,
                   const orc_gains* g, double* f, double* ds_out)
{
    static const double zero[3] = { 0, 0, 0 };
    return pair_force(p, v, c, r, u ? u : zero, g, f, ds_out);
}

/* Eq. 3 alone, for pin P2 (c . n = 0). */
void orc_current_vector(const double* p, const double* v, const double* c, const double* u, double* cur)
{
    double d[3] = { c[0] - p[0], c[1] - p[1], c[2] - p[2] };
    double dist = norm3(d);
    double vr[3] = { v[0] - (u ? u[0] : 0), v[1] - (u ? u[1] : 0), v[2] - (u ? u[2] : 0) };
    double n[3] = { d[0] / dist, d[1] / dist, d[2] / dist };
    double ndv = dot3(n, vr);
    for (int i = 0; i < 3; ++i) cur[i] = vr[i] - n[i] * ndv;
}

/* Sum over the sphere world S_W (Eq. 5-6; Alg. 1's reduction as a plain sequential sum) at
 * obstacle time t (G25: c_j(t) = c_j + t u_j).  Also returns: dmin = min_j ds; sum_mag = sum_j ||f_j||;
 * margins[0] = min_j |ds - r_d| / r_d (gate), margins[1] = min_j |ds - eps| / eps (clamp) (G10);
 * kappa = max over gated j of ||d|| / dO (conditioning). */
static void sphere_sum(const double p[3], const double v[3], int n_sph, const float* xyzr,
                       const float* vel, double t, const orc_gains* g,
                       double f_r[3], double* dmin, double* sum_mag, double margins[2], double* kappa)
{
    f_r[0] = f_r[1] = f_r[2] = 0.0;
    double dm = INFINITY, sm = 0.0, mg = INFINITY, mc = INFINITY, kap = 0.0;
    for (int j = 0; j < n_sph; ++j) {
        double u[3] = { 0, 0, 0 };
        double c[3] = { xyzr[4*j], xyzr[4*j+1], xyzr[4*j+2] };
        double r = xyzr[4*j+3];
        if (vel) {
            u[0] = vel[3*j]; u[1] = vel[3*j+1]; u[2] = vel[3*j+2];
            c[0] += t * u[0]; c[1] += t * u[1]; c[2] += t * u[2];
        }
        double f[3], ds;
        int gated = pair_force(p, v, c, r, u, g, f, &ds);
        if (ds < dm) dm = ds;
        double a = fabs(ds - g->r_influence) / g->r_influence; if (a < mg) mg = a;
        double b = fabs(ds - g->eps_dist) / g->eps_dist;       if (b < mc) mc = b;
        if (gated) {
            f_r[0] += f[0]; f_r[1] += f[1]; f_r[2] += f[2];
            sm += norm3(f);
            double dO = fmax(ds, g->eps_dist);
            double k = (ds + g->r_agent + r) / dO;
            if (k > kap) kap = k;
        }
    }
    *dmin = dm;
    if (sum_mag) *sum_mag = sm;
    if (margins) { margins[0] = mg; margins[1] = mc; }
    if (kappa) *kappa = kap;
}

/* ------------------------------------------------------------------ SE(3) exp / log
 * Eq. 8 and Eq. 11 on the matrix group: twist (phi, rho) in R^6,
 * rotation part first (G13/G14: full coupled SE(3) log, shortest rotation, exp(log(T)) = T).
 *   exp: R = I + A W + B W^2, t = (I + B W + C W^2) rho,  W = hat(phi), th = ||phi||,
 *        A = sin th / th, B = (1 - cos th)/th^2, C = (th - sin th)/th^3.
 *   log: th from R, phi = th n, rho = (I - W/2 + c2 W^2) t, c2 = (1 - (th/2) cot(th/2)) / th^2.
 * Pinned against scipy.linalg.expm / logm of the 4x4 twist matrix (P10). */
void orc_se3_exp(const double* phi, const double* rho, double* R, double* t)
{
    double th = norm3(phi), th2 = th * th, A, B, C;
    if (th < 1e-2) {
        A = 1.0 - th2 / 6.0 + th2 * th2 / 120.0 - th2 * th2 * th2 / 5040.0;
        B = 0.5 - th2 / 24.0 + th2 * th2 / 720.0 - th2 * th2 * th2 / 40320.0;
        C = 1.0 / 6.0 - th2 / 120.0 + th2 * th2 / 5040.0 - th2 * th2 * th2 / 362880.0;
    } else {
        double sh = sin(0.5 * th);
        A = sin(th) / th;
        B = 2.0 * sh * sh / th2;
        C = (th - sin(th)) / (th2 * th);
    }
    double W[9], W2[9];
    hat3(phi, W);
    mat3_mul(W, W, W2);
    double V[9];
    for (int i = 0; i < 9; ++i) {
        double I = (i % 4 == 0) ? 1.0 : 0.0;
        R[i] = I + A * W[i] + B * W2[i];
        V[i] = I + B * W[i] + C * W2[i];
    }
    mat3_vec(V, rho, t);
}

void orc_se3_log(const double* R, const double* t, double* phi, double* rho)
{
    double vee[3] = { 0.5 * (R[7] - R[5]), 0.5 * (R[2] - R[6]), 0.5 * (R[3] - R[1]) };  /* sin(th) n */
    double s = norm3(vee);
    double c = 0.5 * (R[0] + R[4] + R[8] - 1.0);
    double th = atan2(s, c);
    if (th < 1e-8) {
        double k = 1.0 + th * th / 6.0;
        for (int i = 0; i < 3; ++i) phi[i] = k * vee[i];
    } else if (th < M_PI - 1e-6) {
        for (int i = 0; i < 3; ++i) phi[i] = vee[i] * (th / s);
    } else {
        /* th ~ pi: axis from the symmetric part, R + R^T = 2 cos th I + 2(1 - cos th) n n^T */
        double n[3], omc = 1.0 - c;
        for (int i = 0; i < 3; ++i) { double q = (R[4*i] - c) / omc; n[i] = sqrt(q > 0 ? q : 0); }
        int k = (n[0] >= n[1] && n[0] >= n[2]) ? 0 : (n[1] >= n[2] ? 1 : 2);
        for (int i = 0; i < 3; ++i) if (i != k) {
            double sym = 0.5 * (R[3*i+k] + R[3*k+i]) / omc;    /* n_i n_k */
            n[i] = sym / n[k];
        }
        if (dot3(n, vee) < 0) { n[0] = -n[0]; n[1] = -n[1]; n[2] = -n[2]; }
        double nn = norm3(n);
        for (int i = 0; i < 3; ++i) phi[i] = th * n[i] / nn;
    }
    double th2 = th * th, c2;
    if (th < 1e-2) c2 = 1.0 / 12.0 + th2 / 720.0 + th2 * th2 / 30240.0 + th2 * th2 * th2 / 1209600.0;
    else           c2 = (1.0 - 0.5 * th * cos(0.5 * th) / sin(0.5 * th)) / th2;
    double W[9], W2[9], Vi[9];
    hat3(phi, W);
    mat3_mul(W, W, W2);
    for (int i = 0; i < 9; ++i) Vi[i] = ((i % 4 == 0) ? 1.0 : 0.0) - 0.5 * W[i] + c2 * W2[i];
    mat3_vec(Vi, t, rho);
}

/* ------------------------------------------------------------------ per-pose cost pieces */
typedef struct {
    double sumG, sumO, L, J, minclr, d1;
    int collided;
    double hist[4][3];   /* last 4 poses, hist[0] oldest */
    int n_hist;
} cost_acc;

static void cost_init(cost_acc* a, const double p[3], const double goal[3]) {
    memset(a, 0, sizeof *a);
    a->minclr = INFINITY;
    double e[3] = { goal[0] - p[0], goal[1] - p[1], goal[2] - p[2] };
    a->d1 = norm3(e);                                  /* d_min^(1), Eq. 19 */
}
/* Eq. 17 and 18 summands at one pose (G20, G21, G33), collision record (G34). */
static void cost_pose(cost_acc* a, const double p[3], const double goal[3], double dmin, const orc_gains* g) {
    double rcg = g->r_cost_goal > 0 ? g->r_cost_goal : g->r_influence;
    double rco = g->r_cost_obs > 0 ? g->r_cost_obs : g->r_influence;
    double e[3] = { goal[0] - p[0], goal[1] - p[1], goal[2] - p[2] };
    a->sumG += fmin(norm3(e), rcg) / rcg;
    double dc = dmin < 0 ? 0 : (dmin > rco ? rco : dmin);
    a->sumO += 1.0 - dc / rco;
    if (dmin < a->minclr) a->minclr = dmin;
    if (dmin < 0) a->collided = 1;
}
/* Eq. 19's L_path and Eq. 20's J, literally from positions. */
static void cost_move(cost_acc* a, const double p_old[3], const double p_new[3]) {
    double dp[3] = { p_new[0] - p_old[0], p_new[1] - p_old[1], p_new[2] - p_old[2] };
    a->L += norm3(dp);
    if (a->n_hist == 0) { memcpy(a->hist[0], p_old, sizeof(double) * 3); a->n_hist = 1; }
    if (a->n_hist < 4) { memcpy(a->hist[a->n_hist], p_new, sizeof(double) * 3); a->n_hist++; }
    else {
        memmove(a->hist[0], a->hist[1], sizeof(double) * 9);
        memcpy(a->hist[3], p_new, sizeof(double) * 3);
    }
    if (a->n_hist == 4) {
        double s = 0;
        for (int i = 0; i < 3; ++i) {
            double t = a->hist[3][i] - 3.0 * a->hist[2][i] + 3.0 * a->hist[1][i] - a->hist[0][i];
            s += t * t;
        }
        a->J += s;
    }
}
/* Eq. 16-20 final assembly; N_k = steps + 1 poses (G19). out = {C, C_goal, C_obs, C_path, C_smooth}. */
static void cost_finish(const cost_acc* a, int steps, double dt, const orc_gains* g, double out[5]) {
    double Nk = (double)steps + 1.0;
    double Cg = a->sumG / Nk, Co = a->sumO / Nk, Cp, Cs;
    if (a->L == 0.0 && a->d1 == 0.0) Cp = 0.0;
    else if (a->L >= a->d1) Cp = 1.0 - a->d1 / a->L;        /* Eq. 19 first rendering (G22) */
    else Cp = 1.0 - a->L / a->d1;
    Cs = fmin(1.0, a->J / (Nk * dt * dt * dt * dt * g->a_max * g->a_max));   /* Eq. 20 */
    out[1] = Cg; out[2] = Co; out[3] = Cp; out[4] = Cs;
    out[0] = g->w_goal * Cg + g->w_obs * Co + g->w_path * Cp + g->w_smooth * Cs;   /* Eq. 16 */
}

/* ------------------------------------------------------------------ 3D point agents
 * agents [n][6] = (p, v) float32 (the same FP32-rounded inputs the GPU gets), promoted to double.
 * Outputs (any may be NULL): final [n][6]; cost [n][5]; minclr [n]; collided [n];
 * margins [n][3] = min over the rollout of (gate margin, clamp margin, |dmin| clearance margin);
 * traj [n][steps+1][6] = state (p, v) at the START of step k (k = 0..steps-1) and the final state.
 * threads > 1: OpenMP over agents (timing only). */
void orc_rollout_point3(int n_agents, const float* agents, int n_sph, const float* xyzr, const float* vel,
                        const float* goal, const orc_gains* g, double dt, int steps, int threads,
                        double* final, double* cost, double* minclr, int* collided,
                        double* margins, double* traj)
{
    const double pg[3] = { goal[0], goal[1], goal[2] };
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 1 ? threads : 1) if (threads > 1)
#endif
    for (int i = 0; i < n_agents; ++i) {
        double p[3] = { agents[6*i], agents[6*i+1], agents[6*i+2] };
        double v[3] = { agents[6*i+3], agents[6*i+4], agents[6*i+5] };
        cost_acc acc; cost_init(&acc, p, pg);
        double mg = INFINITY, mc = INFINITY, mclr = INFINITY;
        for (int k = 0; k < steps; ++k) {                 /* pose index k+1 */
            double t_k = k * dt;
            if (traj) { double* s = traj + ((size_t)i * (steps + 1) + k) * 6;
                        for (int a = 0; a < 3; ++a) { s[a] = p[a]; s[3+a] = v[a]; } }
            double f_r[3], dmin, m2[2];
            sphere_sum(p, v, n_sph, xyzr, vel, t_k, g, f_r, &dmin, NULL, m2, NULL);
            if (m2[0] < mg) mg = m2[0];
            if (m2[1] < mc) mc = m2[1];
            if (fabs(dmin) < mclr) mclr = fabs(dmin);
            cost_pose(&acc, p, pg, dmin, g);
            double p_new[3];
            for (int a = 0; a < 3; ++a) {
                double f = g->k_att * (pg[a] - p[a]) - g->k_damp * v[a] + f_r[a];  /* Eq. 6-7 */
                double acc_a = g->inv_mass * f;                                    /* Eq. 9 */
                v[a] = v[a] + g->vel_factor * dt * acc_a;                          /* Eq. 10 */
                p_new[a] = p[a] + dt * v[a];                                       /* Eq. 11, point mass (G17) */
            }
            cost_move(&acc, p, p_new);
            p[0] = p_new[0]; p[1] = p_new[1]; p[2] = p_new[2];
        }
        {   /* final pose p^(S+1): distance-only pass (G19) */
            double f_r[3], dmin;
            sphere_sum(p, v, n_sph, xyzr, vel, steps * dt, g, f_r, &dmin, NULL, NULL, NULL);
            if (fabs(dmin) < mclr) mclr = fabs(dmin);
            cost_pose(&acc, p, pg, dmin, g);
            if (traj) { double* s = traj + ((size_t)i * (steps + 1) + steps) * 6;
                        for (int a = 0; a < 3; ++a) { s[a] = p[a]; s[3+a] = v[a]; } }
        }
        if (final) for (int a = 0; a < 3; ++a) { final[6*i+a] = p[a]; final[6*i+3+a] = v[a]; }
        if (cost) cost_finish(&acc, steps, dt, g, cost + 5 * (size_t)i);
        if (minclr) minclr[i] = acc.minclr;
        if (collided) collided[i] = acc.collided;
        if (margins) { margins[3*i] = mg; margins[3*i+1] = mc; margins[3*i+2] = mclr; }
    }
}

/* Forces at given states, no integration (the paper's control-thread query, Fig. 2 step 5,
 * PAPER.md:72, 278).  states [n][6] double.  f_rep, f_total [n][3]; scale [n] = ||f_a|| + sum_j ||f_j||
 * (G29 denominator); margins [n][2]; kappa [n]; dmin [n].  Any output may be NULL. */
void orc_forces_point3(int n, const double* states, int n_sph, const float* xyzr, const float* vel,
                       double t_obstacles, const float* goal, const orc_gains* g,
                       double* f_rep, double* f_total, double* scale, double* margins, double* kappa,
                       double* dmin_out)
{
    for (int i = 0; i < n; ++i) {
        const double* p = states + 6 * (size_t)i;
        const double* v = p + 3;
        double f_r[3], dmin, sm, m2[2], kap, fa[3];
        sphere_sum(p, v, n_sph, xyzr, vel, t_obstacles, g, f_r, &dmin, &sm, m2, &kap);
        for (int a = 0; a < 3; ++a) fa[a] = g->k_att * ((double)goal[a] - p[a]) - g->k_damp * v[a];
        if (f_rep) for (int a = 0; a < 3; ++a) f_rep[3*i+a] = f_r[a];
        if (f_total) for (int a = 0; a < 3; ++a) f_total[3*i+a] = fa[a] + f_r[a];
        if (scale) scale[i] = norm3(fa) + sm;
        if (margins) { margins[2*i] = m2[0]; margins[2*i+1] = m2[1]; }
        if (kappa) kappa[i] = kap;
        if (dmin_out) dmin_out[i] = dmin;
    }
}

/* ------------------------------------------------------------------ 6D pose agents
 * State per agent: R [9] row-major in SO(3), p [3] world, twist [6] = (omega, nu) BODY frame
 * (Eq. 11 right-multiplies, G17).  Matrix representation on purpose: the CUDA path uses 8-float
 * motors, a different representation of the same group Spin(3) |x R^3.
 * One step (Eq. 6-11):
 *   pdot = R nu;  f_r = sphere sum at (p, pdot)           ("pure linear repulsive forces"; G18)
 *   e = log(T^-1 T_g)                                     (Eq. 8)
 *   wrench = (k_att_rot e_w - k_damp_rot omega,  k_att e_v - k_damp nu + R^T f_r)   (Eq. 6-7, G13)
 *   twist += vel_factor dt (inv_inertia tau, inv_mass f)  (Eq. 9-10)
 *   T <- T exp(dt twist)                                  (Eq. 11)
 * Costs use positions only.
 * traj [n][steps+1][18] = (R, p, twist) at the start of each step and the final state. */
static void pose6_wrench(const double R[9], const double p[3], const double tw[6], const double f_r[3],
                         const double Rg[9], const double pg[3], const orc_gains* g, double wrench[6], double e[6])
{
    double Rrel[9], Rt[9], dp[3] = { pg[0] - p[0], pg[1] - p[1], pg[2] - p[2] }, trel[3], fb[3];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Rt[3*i+j] = R[3*j+i];
    mat3_mul(Rt, Rg, Rrel);
    mat3T_vec(R, dp, trel);
    orc_se3_log(Rrel, trel, e, e + 3);
    mat3T_vec(R, f_r, fb);
    for (int a = 0; a < 3; ++a) {
        wrench[a] = g->k_att_rot * e[a] - g->k_damp_rot * tw[a];
        wrench[3+a] = g->k_att * e[3+a] - g->k_damp * tw[3+a] + fb[a];
    }
}

void orc_rollout_pose6(int n_agents, const double* R0, const double* p0, const double* twist0,
                       int n_sph, const float* xyzr, const float* vel,
                       const double* goal_R, const double* goal_p, const orc_gains* g,
                       double dt, int steps, int threads,
                       double* R_out, double* p_out, double* twist_out,
                       double* cost, double* minclr, int* collided, double* margins, double* traj)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 1 ? threads : 1) if (threads > 1)
#endif
    for (int i = 0; i < n_agents; ++i) {
        double R[9], p[3], tw[6];
        memcpy(R, R0 + 9 * (size_t)i, sizeof R);
        memcpy(p, p0 + 3 * (size_t)i, sizeof p);
        memcpy(tw, twist0 + 6 * (size_t)i, sizeof tw);
        cost_acc acc; cost_init(&acc, p, goal_p);
        double mg = INFINITY, mc = INFINITY, mclr = INFINITY;
        for (int k = 0; k <= steps; ++k) {
            if (traj) { double* s = traj + ((size_t)i * (steps + 1) + k) * 18;
                        memcpy(s, R, sizeof R); memcpy(s + 9, p, sizeof p); memcpy(s + 12, tw, sizeof tw); }
            double pdot[3], f_r[3], dmin, m2[2];
            mat3_vec(R, tw + 3, pdot);
            sphere_sum(p, pdot, n_sph, xyzr, vel, k * dt, g, f_r, &dmin, NULL, m2, NULL);
            if (fabs(dmin) < mclr) mclr = fabs(dmin);
            cost_pose(&acc, p, goal_p, dmin, g);
            if (k == steps) break;                       /* final pose: distance-only (G19) */
            if (m2[0] < mg) mg = m2[0];
            if (m2[1] < mc) mc = m2[1];
            double wrench[6], e[6];
            pose6_wrench(R, p, tw, f_r, goal_R, goal_p, g, wrench, e);
            for (int a = 0; a < 3; ++a) {
                tw[a]   += g->vel_factor * dt * g->inv_inertia * wrench[a];       /* Eq. 9-10 */
                tw[3+a] += g->vel_factor * dt * g->inv_mass * wrench[3+a];
            }
            double phi[3] = { dt * tw[0], dt * tw[1], dt * tw[2] };
            double rho[3] = { dt * tw[3], dt * tw[4], dt * tw[5] };
            double Rd[9], td[3], Rn[9], wd[3], p_new[3];
            orc_se3_exp(phi, rho, Rd, td);                                         /* Eq. 11 */
            mat3_vec(R, td, wd);
            for (int a = 0; a < 3; ++a) p_new[a] = p[a] + wd[a];
            mat3_mul(R, Rd, Rn);
            cost_move(&acc, p, p_new);
            memcpy(R, Rn, sizeof R);
            memcpy(p, p_new, sizeof p);
        }
        if (R_out) memcpy(R_out + 9 * (size_t)i, R, sizeof R);
        if (p_out) memcpy(p_out + 3 * (size_t)i, p, sizeof p);
        if (twist_out) memcpy(twist_out + 6 * (size_t)i, tw, sizeof tw);
        if (cost) cost_finish(&acc, steps, dt, g, cost + 5 * (size_t)i);
        if (minclr) minclr[i] = acc.minclr;
        if (collided) collided[i] = acc.collided;
        if (margins) { margins[3*i] = mg; margins[3*i+1] = mc; margins[3*i+2] = mclr; }
    }
}

/* Forces / wrenches at given 6D states.  f_rep [n][3] world; wrench [n][6] body (tau, f);
 * scale [n] = ||K e - D v|| (6-norm) + sum_j ||f_j||; err [n][6] = the log-map error e (Eq. 8). */
void orc_forces_pose6(int n, const double* R, const double* p, const double* twist,
                      int n_sph, const float* xyzr, const float* vel, double t_obstacles,
                      const double* goal_R, const double* goal_p, const orc_gains* g,
                      double* f_rep, double* wrench_out, double* scale, double* margins, double* err)
{
    static const double zero3[3] = { 0, 0, 0 };
    for (int i = 0; i < n; ++i) {
        const double* Ri = R + 9 * (size_t)i; const double* pi = p + 3 * (size_t)i;
        const double* tw = twist + 6 * (size_t)i;
        double pdot[3], f_r[3], dmin, sm, m2[2], kap, w[6], wa[6], e[6];
        mat3_vec(Ri, tw + 3, pdot);
        sphere_sum(pi, pdot, n_sph, xyzr, vel, t_obstacles, g, f_r, &dmin, &sm, m2, &kap);
        pose6_wrench(Ri, pi, tw, f_r, goal_R, goal_p, g, w, e);
        pose6_wrench(Ri, pi, tw, zero3, goal_R, goal_p, g, wa, e);
        if (f_rep) for (int a = 0; a < 3; ++a) f_rep[3*i+a] = f_r[a];
        if (wrench_out) for (int a = 0; a < 6; ++a) wrench_out[6*i+a] = w[a];
        if (scale) { double s = 0; for (int a = 0; a < 6; ++a) s += wa[a] * wa[a]; scale[i] = sqrt(s) + sm; }
        if (margins) { margins[2*i] = m2[0]; margins[2*i+1] = m2[1]; }
        if (err) for (int a = 0; a < 6; ++a) err[6*i+a] = e[a];
    }
}

/* ------------------------------------------------------------------ selection (G24)
 * Lexicographic argmin of (collided, C, index); a NaN cost ranks as collided with C = +inf.
 * Hysteresis: the incumbent prev_best keeps its place unless the challenger is collision-free
 * while the incumbent collided, or flags are equal and C_best < alpha * C_prev. */
int orc_best_agent(int n, const double* cost5, const int* collided, double alpha, int prev_best, double* out_cost)
{
    int best = -1, bc = 2; double bC = INFINITY;
    for (int i = 0; i < n; ++i) {
        double C = cost5[5 * (size_t)i]; int cf = collided[i] ? 1 : 0;
        if (C != C) { C = INFINITY; cf = 1; }
        if (best < 0 || cf < bc || (cf == bc && C < bC)) { best = i; bc = cf; bC = C; }
    }
    if (best >= 0 && prev_best >= 0 && prev_best < n && prev_best != best) {
        double Cp = cost5[5 * (size_t)prev_best]; int cp = collided[prev_best] ? 1 : 0;
        if (Cp != Cp) { Cp = INFINITY; cp = 1; }
        int improves = (bc < cp) || (bc == cp && bC < alpha * Cp);
        if (!improves) { best = prev_best; bC = Cp; }
    }
    if (out_cost) *out_cost = best >= 0 ? bC : NAN;
    return best;
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
