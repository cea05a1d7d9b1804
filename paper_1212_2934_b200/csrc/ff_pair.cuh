// ff_pair.cuh -- Eq. 11 (field) and Eq. 12 (force) pair terms in packed FP32.
//
// sm_100 has packed FP32 instructions (FFMA2 / FMUL2 / FADD2, reached through __ffma2_rn,
// __fmul2_rn, __fadd2_rn).  One lane evaluates ONE source against TWO targets per instruction:
// the target-side values are register pairs (.x = first target, .y = second target) and the
// source-side values are scalars, which the packed instructions take in their broadcast operand
// form (`R.F32`), so a source costs six 32-bit words of shared-memory traffic for two interactions:
//   A = x, y, z, mx        B = my, mz            (one 32-byte ring / tile record per source)
// Why this way round: the register file delivers one even and one odd register per lane and cycle,
// a packed instruction with three register-PAIR operands therefore issues every 3 cycles instead of
// every 2; with scalar source operands fewer instructions are of that form than with the sources
// packed in pairs (measured: 95 against 99.5 cycles per 64 interactions, ff_measure_probe).
// Used by the tree walk (ff_walk.cu), the tiled all-pairs kernel (ff_direct.cu) and the probe
// (ff_probe.cu).
#pragma once
#include <cuda_runtime.h>

__device__ __forceinline__ float2 ff_dup(float a) { return make_float2(a, a); }

// MUFU.RSQ without the denormal pre/post-scaling of rsqrtf (2 FSETP + 4 FMUL per pair of sources):
// r^2 of two distinct particles is never denormal for inputs the ABI allows.
__device__ __forceinline__ float ff_rsqrt(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float2 ff_rsqrt2(float2 r2) { return make_float2(ff_rsqrt(r2.x), ff_rsqrt(r2.y)); }

// the two targets of one lane: position and moment, .x = first target, .y = second target
struct ff_target2 {
    float2 px, py, pz, ux, uy, uz;
};

// A register PAIR the compiler cannot rebuild from its two halves later on: without this ptxas keeps the two targets'
// values in the registers they were loaded into and re-assembles the pairs with two MOVs per use inside the
// evaluation loop (measured: +11 % instructions).  The volatile asm is opaque and cannot be duplicated.
__device__ __forceinline__ float2 ff_pin_pair(float a, float b)
{
    unsigned long long v;
    asm volatile("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(a), "f"(b));
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}

// running sums of one lane for its two targets; f = fv + sk u_k (the u_k term of Eq. 12 is
// accumulated as a scalar and applied once at the end).  The two parts of Eq. 11 go into ONE
// accumulator: for aligned moments sum 3 rho (u.rho)/r^5 and sum u/r^3 are each far larger than
// their difference, and separate fp32 sums would lose that difference to rounding.
struct ff_acc2 {
    float2 hx, hy, hz, fx, fy, fz, sk;
};
__device__ __forceinline__ void ff_acc2_zero(ff_acc2& s) { s.hx = s.hy = s.hz = s.fx = s.fy = s.fz = s.sk = ff_dup(0.0f); }

// rho = p_k - p_j for both targets (one rounding, as a subtraction) and r^2
__device__ __forceinline__ void ff_pair2_geom(const float4& A, const ff_target2& t, float2& dx, float2& dy, float2& dz,
                                              float2& r2)
{
    const float2 neg1 = ff_dup(-1.0f);
    dx = __ffma2_rn(ff_dup(A.x), neg1, t.px);
    dy = __ffma2_rn(ff_dup(A.y), neg1, t.py);
    dz = __ffma2_rn(ff_dup(A.z), neg1, t.pz);
    r2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
}

// One source term of Eq. 11 (h) and Eq. 12 (f) for two targets.  rinv = 1/|rho| per target (0 for a
// term that is to be skipped):
//   h_kj = 3 rho (u_j.rho)/r^5 - u_j/r^3
//   f_kj = { rho [(u_j.u_k) - 5 (u_j.rho)(u_k.rho)/r^2] + u_k (u_j.rho) + u_j (u_k.rho) } 3/r^5
// 38 packed FP32 instructions + 2 MUFU.RSQ per source and target pair (ff_pair2_geom included).
// EXTRA: `extra` is added to the coefficient of rho in f (the all-pairs MD step puts the Lennard-Jones term of
// Eq. 13 there: f^sr_kj = w rho with w = 24 eps [ (s/r)^12 - (s/r)^6 ] / r^2, PAPER.md:74 and Algorithm 1 line 8)
template <bool EXTRA = false>
__device__ __forceinline__ void ff_pair2_accum(const float4& A, const float2& B, const ff_target2& t, float2 dx, float2 dy,
                                               float2 dz, float2 rinv, ff_acc2& s, float2 extra = make_float2(0.f, 0.f))
{
    const float2 mx = ff_dup(A.w), my = ff_dup(B.x), mz = ff_dup(B.y);
    const float2 rinv2 = __fmul2_rn(rinv, rinv);
    const float2 nr3 = __fmul2_rn(rinv2, make_float2(-rinv.x, -rinv.y));           // -1 / r^3 (negation folds into the operand)
    const float2 r5 = __fmul2_rn(nr3, __fmul2_rn(rinv2, ff_dup(-3.0f)));           // 3 / r^5 = (-1/r^3)(-3/r^2)
    const float2 a = __ffma2_rn(mz, dz, __ffma2_rn(my, dy, __fmul2_rn(mx, dx)));   // u_j . rho
    const float2 b = __ffma2_rn(t.uz, dz, __ffma2_rn(t.uy, dy, __fmul2_rn(t.ux, dx)));   // u_k . rho
    const float2 c = __ffma2_rn(mz, t.uz, __ffma2_rn(my, t.uy, __fmul2_rn(mx, t.ux)));   // u_j . u_k
    const float2 ca = __fmul2_rn(a, r5);
    const float2 cb = __fmul2_rn(b, r5);
    s.hx = __ffma2_rn(ca, dx, s.hx); s.hy = __ffma2_rn(ca, dy, s.hy); s.hz = __ffma2_rn(ca, dz, s.hz);
    s.hx = __ffma2_rn(nr3, mx, s.hx); s.hy = __ffma2_rn(nr3, my, s.hy); s.hz = __ffma2_rn(nr3, mz, s.hz);
    const float2 w = __fmul2_rn(__fmul2_rn(ca, b), rinv2);                         // 3 (u_j.rho)(u_k.rho) / r^7
    float2 cr = __ffma2_rn(ff_dup(-5.0f), w, __fmul2_rn(c, r5));
    if (EXTRA) cr = __fadd2_rn(cr, extra);
    s.fx = __ffma2_rn(cr, dx, s.fx); s.fy = __ffma2_rn(cr, dy, s.fy); s.fz = __ffma2_rn(cr, dz, s.fz);
    s.fx = __ffma2_rn(cb, mx, s.fx); s.fy = __ffma2_rn(cb, my, s.fy); s.fz = __ffma2_rn(cb, mz, s.fz);
    s.sk = __fadd2_rn(s.sk, ca);
}

// one source against the lane's two targets, nothing masked (the hot loop of the walk and of the direct kernel)
__device__ __forceinline__ void ff_pair2(const float4& A, const float2& B, const ff_target2& t, ff_acc2& s)
{
    float2 dx, dy, dz, r2;
    ff_pair2_geom(A, t, dx, dy, dz, r2);
    ff_pair2_accum(A, B, t, dx, dy, dz, ff_rsqrt2(r2), s);
}
