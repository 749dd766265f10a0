// gmapp_microbench.cuh -- issue-cost microbenchmarks behind the instruction-mix reasoning of DESIGN.md section 6
// (gmapp_microbench in include/gmapp.h; results recorded in profiles/r02_microbench.md).  Register-only kernels: every
// SM runs one 512-thread CTA (4 warps per SM sub-partition), each thread `iters` rounds of 8 independent chains of ONE
// instruction kind; reported: SM cycles per warp-instruction per sub-partition = time x clock / (4 warps x iters x 8).
// Compiled in gmapp.cu only.
#pragma once
#include <cuda_runtime.h>

namespace gmapp {

enum MicroKind {
    MB_FFMA_3REG = 0,        // fma.rn.f32 x, x, a, b            three distinct registers
    MB_FFMA2_3OP = 1,        // fma.rn.f32x2 X, X, A, B          three distinct register pairs
    MB_FFMA2_2OP = 2,        // fma.rn.f32x2 X, X, X, B          two distinct register pairs
    MB_FFMA2_BCAST = 3,      // fma.rn.f32x2 X, X, {a,a}, B      the broadcast operand form of the sweeps
    MB_MUFU_RCP = 4,         // rcp.approx.ftz.f32 (+ one FADD per MUFU so that ptxas cannot fold rcp(rcp(x)); it co-issues)
    MB_MUFU_RCP_PRED_OFF = 5,// @p rcp.approx.ftz.f32 with p false on every lane
    MB_FMNMX = 6,            // max.f32 (2 inputs)
    MB_FMNMX3 = 7,           // min.f32 (3 inputs)
    MB_FSETP_FSEL = 8,       // setp.gt.f32 + selp.f32 (two instructions per chain step: the reported cost is per PAIR)
    MB_FFMA2_3OP_NOREUSE = 9,// fma.rn.f32x2 X_i, X_i, Y_i, Z_i  three distinct register pairs, none shared between chains
    MB_FFMA2_FMNMX = 10,     // one FFMA2 + one FMNMX on separate chains (cost per PAIR): 2.03 if the ALU op co-issues, 3.06 if not
    MB_FFMA2_2FMNMX = 11,    // one FFMA2 + two FMNMX (per triple)
    MB_FFMA_FMNMX = 12,      // one scalar FFMA + one FMNMX (per pair)
    MB_SWEEP_MIX = 13,       // the raw sweep's mix per agent-trip: 16 FFMA2, 4 MUFU, 5 FMNMX, 2 FSETP+FSEL (cost per group of 29)
    MB_SWEEP_MIX_SCALAR = 14,// the same mix with 32 scalar FFMA in place of the 16 FFMA2 (cost per group of 45)
    MB_COUNT = 15
};

template <int KIND>
__global__ void __launch_bounds__(512) k_microbench(float* out, int iters, float a, float b, float thr) {
    float x[8];
    unsigned long long X[8], Y[8], Z[8], A, B;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        x[i] = 0.5f + float(threadIdx.x + 37 * i) * 1e-4f;
        asm("mov.b64 %0, {%1, %2};" : "=l"(X[i]) : "f"(x[i]), "f"(x[i] + 0.25f));
        asm("mov.b64 %0, {%1, %2};" : "=l"(Y[i]) : "f"(a - 1e-4f * i), "f"(a - 2e-4f * i));
        asm("mov.b64 %0, {%1, %2};" : "=l"(Z[i]) : "f"(b + 1e-5f * i), "f"(b + 2e-5f * i));
    }
    asm("mov.b64 %0, {%1, %2};" : "=l"(A) : "f"(a), "f"(a * 0.999f));
    asm("mov.b64 %0, {%1, %2};" : "=l"(B) : "f"(b), "f"(b * 1.001f));
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (KIND == MB_FFMA_3REG) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[i]) : "f"(a), "f"(b));
            if (KIND == MB_FFMA2_3OP) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(X[i]) : "l"(A), "l"(B));
            if (KIND == MB_FFMA2_2OP) asm volatile("fma.rn.f32x2 %0, %0, %0, %1;" : "+l"(X[i]) : "l"(B));
            if (KIND == MB_FFMA2_BCAST) asm volatile("{ .reg .b64 t; mov.b64 t, {%1, %1}; fma.rn.f32x2 %0, %0, t, %2; }" : "+l"(X[i]) : "f"(a), "l"(B));
            if (KIND == MB_MUFU_RCP) asm volatile("{ .reg .f32 t; rcp.approx.ftz.f32 t, %0; add.f32 %0, t, %1; }" : "+f"(x[i]) : "f"(b));
            if (KIND == MB_FFMA2_3OP_NOREUSE) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(X[i]) : "l"(Y[i]), "l"(Z[i]));
            if (KIND == MB_MUFU_RCP_PRED_OFF) asm volatile("{ .reg .pred p; setp.gt.f32 p, %0, %1; @p rcp.approx.ftz.f32 %0, %0; }" : "+f"(x[i]) : "f"(thr));
            if (KIND == MB_FMNMX) asm volatile("max.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(a));
            if (KIND == MB_FMNMX3) asm volatile("min.f32 %0, %0, %1, %2;" : "+f"(x[i]) : "f"(a), "f"(b));
            if (KIND == MB_FFMA2_FMNMX) {
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(X[i]) : "l"(A), "l"(B));
                asm volatile("max.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(a));
            }
            if (KIND == MB_FFMA2_2FMNMX) {
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(X[i]) : "l"(A), "l"(B));
                asm volatile("max.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(a));
                asm volatile("min.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(b));
            }
            if (KIND == MB_FFMA_FMNMX) {
                float lo, hi;
                asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(X[i]));
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(lo) : "f"(a), "f"(b));
                asm volatile("mov.b64 %0, {%1, %2};" : "=l"(X[i]) : "f"(lo), "f"(hi));
                asm volatile("max.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(a));
            }
            if (KIND == MB_SWEEP_MIX && (i & 1) == 0) {      // 4 groups per round; chains: X[i], X[i+1] packed; x[i], x[i+1] scalar
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(X[i]) : "l"(A), "l"(B));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(X[i + 1]) : "l"(A), "l"(B));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(Y[i]) : "l"(A), "l"(B));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(Y[i + 1]) : "l"(A), "l"(B));
                asm volatile("{ .reg .f32 t; rsqrt.approx.ftz.f32 t, %0; max.f32 %0, t, %1; }" : "+f"(x[i]) : "f"(a));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(Z[i]) : "l"(A), "l"(B));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(Z[i + 1]) : "l"(A), "l"(B));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(X[i]) : "l"(A), "l"(B));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(X[i + 1]) : "l"(A), "l"(B));
                asm volatile("{ .reg .f32 t; rsqrt.approx.ftz.f32 t, %0; max.f32 %0, t, %1; }" : "+f"(x[i + 1]) : "f"(a));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(Y[i]) : "l"(A), "l"(B));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(Y[i + 1]) : "l"(A), "l"(B));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(Z[i]) : "l"(A), "l"(B));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(Z[i + 1]) : "l"(A), "l"(B));
                asm volatile("{ .reg .f32 t; .reg .pred p; rcp.approx.ftz.f32 t, %0; min.f32 t, t, %1, %2; setp.gt.f32 p, t, %3; selp.f32 %0, %1, t, p; }" : "+f"(x[i]) : "f"(a), "f"(b), "f"(thr));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(X[i]) : "l"(A), "l"(B));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(X[i + 1]) : "l"(A), "l"(B));
                asm volatile("{ .reg .f32 t; .reg .pred p; rcp.approx.ftz.f32 t, %0; max.f32 t, t, %1; setp.gt.f32 p, t, %3; selp.f32 %0, %2, t, p; }" : "+f"(x[i + 1]) : "f"(a), "f"(b), "f"(thr));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(Y[i]) : "l"(A), "l"(B));
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(Y[i + 1]) : "l"(A), "l"(B));
            }
            if (KIND == MB_SWEEP_MIX_SCALAR && (i & 1) == 0) {
                float lo[6], hi[6];
                asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(lo[0]), "=f"(hi[0]) : "l"(X[i]));
                asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(lo[1]), "=f"(hi[1]) : "l"(X[i + 1]));
                asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(lo[2]), "=f"(hi[2]) : "l"(Y[i]));
                asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(lo[3]), "=f"(hi[3]) : "l"(Y[i + 1]));
                asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(lo[4]), "=f"(hi[4]) : "l"(Z[i]));
                asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(lo[5]), "=f"(hi[5]) : "l"(Z[i + 1]));
#define MB_F2(k) asm volatile("fma.rn.f32 %0, %0, %2, %3; fma.rn.f32 %1, %1, %2, %3;" : "+f"(lo[k]), "+f"(hi[k]) : "f"(a), "f"(b));
                MB_F2(0) MB_F2(1) MB_F2(2) MB_F2(3)
                asm volatile("{ .reg .f32 t; rsqrt.approx.ftz.f32 t, %0; max.f32 %0, t, %1; }" : "+f"(x[i]) : "f"(a));
                MB_F2(4) MB_F2(5) MB_F2(0) MB_F2(1)
                asm volatile("{ .reg .f32 t; rsqrt.approx.ftz.f32 t, %0; max.f32 %0, t, %1; }" : "+f"(x[i + 1]) : "f"(a));
                MB_F2(2) MB_F2(3) MB_F2(4) MB_F2(5)
                asm volatile("{ .reg .f32 t; .reg .pred p; rcp.approx.ftz.f32 t, %0; min.f32 t, t, %1, %2; setp.gt.f32 p, t, %3; selp.f32 %0, %1, t, p; }" : "+f"(x[i]) : "f"(a), "f"(b), "f"(thr));
                MB_F2(0) MB_F2(1)
                asm volatile("{ .reg .f32 t; .reg .pred p; rcp.approx.ftz.f32 t, %0; max.f32 t, t, %1; setp.gt.f32 p, t, %3; selp.f32 %0, %2, t, p; }" : "+f"(x[i + 1]) : "f"(a), "f"(b), "f"(thr));
                MB_F2(2) MB_F2(3)
#undef MB_F2
                asm volatile("mov.b64 %0, {%1, %2};" : "=l"(X[i]) : "f"(lo[0]), "f"(hi[0]));
                asm volatile("mov.b64 %0, {%1, %2};" : "=l"(X[i + 1]) : "f"(lo[1]), "f"(hi[1]));
                asm volatile("mov.b64 %0, {%1, %2};" : "=l"(Y[i]) : "f"(lo[2]), "f"(hi[2]));
                asm volatile("mov.b64 %0, {%1, %2};" : "=l"(Y[i + 1]) : "f"(lo[3]), "f"(hi[3]));
                asm volatile("mov.b64 %0, {%1, %2};" : "=l"(Z[i]) : "f"(lo[4]), "f"(hi[4]));
                asm volatile("mov.b64 %0, {%1, %2};" : "=l"(Z[i + 1]) : "f"(lo[5]), "f"(hi[5]));
            }
            if (KIND == MB_FSETP_FSEL) asm volatile("{ .reg .pred p; setp.gt.f32 p, %0, %1; selp.f32 %0, %2, %0, p; }" : "+f"(x[i]) : "f"(thr), "f"(a));
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < 8; ++i) { float lo, hi; asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(X[i])); s += x[i] + lo + hi; }
    if (KIND == MB_FFMA2_3OP_NOREUSE || KIND == MB_SWEEP_MIX || KIND == MB_SWEEP_MIX_SCALAR) {
#pragma unroll
        for (int i = 0; i < 8; ++i) { float lo, hi; asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(Y[i] ^ Z[i])); s += lo + hi; }
    }
    if (s == 123.456f) out[0] = s;      // never true in practice; keeps the chains alive
}

}  // namespace gmapp
