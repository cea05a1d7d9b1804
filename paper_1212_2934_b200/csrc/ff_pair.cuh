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
// (the vector form: used with the first-order cell term below, which needs u_k.rho anyway; the walk's and the
// all-pairs kernel's main loops use the tensor form further down)
__device__ __forceinline__ void ff_pair2_accum(const float4& A, const float2& B, const ff_target2& t, float2 dx, float2 dy,
                                               float2 dz, float2 rinv, ff_acc2& s)
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
    const float2 cr = __ffma2_rn(ff_dup(-5.0f), w, __fmul2_rn(c, r5));
    s.fx = __ffma2_rn(cr, dx, s.fx); s.fy = __ffma2_rn(cr, dy, s.fy); s.fz = __ffma2_rn(cr, dz, s.fz);
    s.fx = __ffma2_rn(cb, mx, s.fx); s.fy = __ffma2_rn(cb, my, s.fy); s.fz = __ffma2_rn(cb, mz, s.fz);
    s.sk = __fadd2_rn(s.sk, ca);
}


// ---- the same pair terms with the force kept as a TENSOR ---------------------------------------------------------
// Eq. 12 is linear in the target's moment: f_k = G u_k with the symmetric, traceless field-gradient tensor
//     G = sum_j { p (rho (x) u_j + u_j (x) rho + a 1) + q rho (x) rho },   p = 3/r^5, a = u_j.rho, q = -5 p a / r^2
//       = sum_j { (p rho) (x) e + e (x) (p rho) + p a 1 },                 e = u_j - 2.5 (a / r^2) rho
// so the target's moment leaves the loop: no u_k.rho, no u_j.u_k, and the nine sums h (3), T_aa = sum (p rho_a) e_a (3),
// G_ab (3 off-diagonal) are applied to u_k once at the end.  The diagonal needs no sum of its own: the tensor is
// traceless term by term (rho.e = -1.5 a), so sum_j p a = -(2/3)(Txx + Tyy + Tzz).
// 36 packed FP32 instructions + 2 MUFU.RSQ per source and target pair (38 with the vector form above).
struct ff_accg2 {
    float2 hx, hy, hz, txx, tyy, tzz, gxy, gxz, gyz;
};
__device__ __forceinline__ void ff_accg2_zero(ff_accg2& s)
{
    s.hx = s.hy = s.hz = s.txx = s.tyy = s.tzz = s.gxy = s.gxz = s.gyz = ff_dup(0.0f);
}

__device__ __forceinline__ void ff_pair2g_accum(const float4& A, const float2& B, float2 dx, float2 dy, float2 dz,
                                                float2 rinv, ff_accg2& s)
{
    const float2 mx = ff_dup(A.w), my = ff_dup(B.x), mz = ff_dup(B.y);
    const float2 rinv2 = __fmul2_rn(rinv, rinv);
    const float2 nr3 = __fmul2_rn(rinv2, make_float2(-rinv.x, -rinv.y));           // -1 / r^3
    const float2 p = __fmul2_rn(nr3, __fmul2_rn(rinv2, ff_dup(-3.0f)));            // 3 / r^5
    const float2 a = __ffma2_rn(mz, dz, __ffma2_rn(my, dy, __fmul2_rn(mx, dx)));   // u_j . rho
    const float2 px = __fmul2_rn(p, dx), py = __fmul2_rn(p, dy), pz = __fmul2_rn(p, dz);   // p rho
    s.hx = __ffma2_rn(px, a, s.hx); s.hy = __ffma2_rn(py, a, s.hy); s.hz = __ffma2_rn(pz, a, s.hz);
    s.hx = __ffma2_rn(nr3, mx, s.hx); s.hy = __ffma2_rn(nr3, my, s.hy); s.hz = __ffma2_rn(nr3, mz, s.hz);
    const float2 m = __fmul2_rn(a, __fmul2_rn(rinv2, ff_dup(-2.5f)));              // -2.5 a / r^2
    const float2 ex = __ffma2_rn(m, dx, mx), ey = __ffma2_rn(m, dy, my), ez = __ffma2_rn(m, dz, mz);
    s.txx = __ffma2_rn(px, ex, s.txx); s.tyy = __ffma2_rn(py, ey, s.tyy); s.tzz = __ffma2_rn(pz, ez, s.tzz);
    s.gxy = __ffma2_rn(px, ey, s.gxy); s.gxy = __ffma2_rn(py, ex, s.gxy);
    s.gxz = __ffma2_rn(px, ez, s.gxz); s.gxz = __ffma2_rn(pz, ex, s.gxz);
    s.gyz = __ffma2_rn(py, ez, s.gyz); s.gyz = __ffma2_rn(pz, ey, s.gyz);
}

// f = G u for the lane's two targets: G_aa = 2 T_aa + S with S = sum_j p a = -(2/3) tr T, off-diagonals as summed
__device__ __forceinline__ void ff_accg2_apply(const ff_accg2& s, float2 ux, float2 uy, float2 uz, float2& fx, float2& fy,
                                               float2& fz)
{
    const float2 S = __fmul2_rn(__fadd2_rn(__fadd2_rn(s.txx, s.tyy), s.tzz), ff_dup(-2.0f / 3.0f));
    const float2 two = ff_dup(2.0f);
    const float2 gxx = __ffma2_rn(two, s.txx, S), gyy = __ffma2_rn(two, s.tyy, S), gzz = __ffma2_rn(two, s.tzz, S);
    fx = __ffma2_rn(s.gxz, uz, __ffma2_rn(s.gxy, uy, __fmul2_rn(gxx, ux)));
    fy = __ffma2_rn(s.gyz, uz, __ffma2_rn(gyy, uy, __fmul2_rn(s.gxy, ux)));
    fz = __ffma2_rn(gzz, uz, __ffma2_rn(s.gyz, uy, __fmul2_rn(s.gxz, ux)));
}

__device__ __forceinline__ void ff_pair2g(const float4& A, const float2& B, const ff_target2& t, ff_accg2& s)
{
    float2 dx, dy, dz, r2;
    ff_pair2_geom(A, t, dx, dy, dz, r2);
    ff_pair2g_accum(A, B, dx, dy, dz, ff_rsqrt2(r2), s);
}

// ---- first-order cell term (FF_OPT_CELL_ORDER = 1) -------------------------
// An accepted cell acts as its pseudo-particle (u', rho') PLUS the next term of the expansion of Eq. 11-12 about
// rho', with the symmetric cell tensor D = sym sum_i (rho_i - rho') (x) u_i.  With R = rho_k - rho', t = tr D,
// b = u_k.R, q = R.D.R, c1 = 3/R^5, c2 = 15/R^7, c3 = 105/R^9 the contracted first-order terms are
//     dh = e R - 2 c1 D R,                                  e = c2 q - c1 t
//     df = g R + 2 c2 b D R + e u_k - 2 (c1 D) u_k,         g = c2 (2 u_k.D.R + t b) - c3 b q
// e u_k joins the scalar accumulator sk of the base term; sum_j c1 D_j is accumulated as a tensor and applied to u_k
// once at the end.  49 more packed FP32 instructions per source and pair of targets.
struct ff_accq2 {
    float2 gxx, gyy, gzz, gxy, gxz, gyz;
};
__device__ __forceinline__ void ff_accq2_zero(ff_accq2& s) { s.gxx = s.gyy = s.gzz = s.gxy = s.gxz = s.gyz = ff_dup(0.0f); }

// Q0 = Dxx, Dyy, Dzz, Dxy ; Q1 = Dxz, Dyz.  A particle carries D = 0: every first-order term is then exactly zero, and
// the 49 instructions are skipped.  The ring entry, and with it this branch, is the same for all lanes that evaluate
// it (a half-warp at W = 32); the walk appends a round's cells before its particles so that the two half-warps mostly
// see the same kind of entry (ff_walk.cu).
__device__ __forceinline__ void ff_pair2_quad(const float4& A, const float2& B, const float4& Q0, const float2& Q1,
                                              const ff_target2& t, ff_acc2& s, ff_accq2& sq)
{
    float2 dx, dy, dz, r2;
    ff_pair2_geom(A, t, dx, dy, dz, r2);
    const float2 rinv = ff_rsqrt2(r2);
    ff_pair2_accum(A, B, t, dx, dy, dz, rinv, s);
    const unsigned any = __float_as_uint(Q0.x) | __float_as_uint(Q0.y) | __float_as_uint(Q0.z) | __float_as_uint(Q0.w) |
                         __float_as_uint(Q1.x) | __float_as_uint(Q1.y);
    if ((any << 1) == 0u) return;                                                  // D = +-0 in all six components
    const float2 rinv2 = __fmul2_rn(rinv, rinv);
    const float2 nr3 = __fmul2_rn(rinv2, make_float2(-rinv.x, -rinv.y));
    const float2 c1 = __fmul2_rn(nr3, __fmul2_rn(rinv2, ff_dup(-3.0f)));           // 3 / R^5
    const float2 c2 = __fmul2_rn(__fmul2_rn(c1, rinv2), ff_dup(5.0f));             // 15 / R^7
    const float2 c3 = __fmul2_rn(__fmul2_rn(c2, rinv2), ff_dup(7.0f));             // 105 / R^9
    const float2 b = __ffma2_rn(t.uz, dz, __ffma2_rn(t.uy, dy, __fmul2_rn(t.ux, dx)));
    const float2 Dxx = ff_dup(Q0.x), Dyy = ff_dup(Q0.y), Dzz = ff_dup(Q0.z), Dxy = ff_dup(Q0.w), Dxz = ff_dup(Q1.x),
                 Dyz = ff_dup(Q1.y);
    const float2 vx = __ffma2_rn(Dxz, dz, __ffma2_rn(Dxy, dy, __fmul2_rn(Dxx, dx)));   // D R
    const float2 vy = __ffma2_rn(Dyz, dz, __ffma2_rn(Dyy, dy, __fmul2_rn(Dxy, dx)));
    const float2 vz = __ffma2_rn(Dzz, dz, __ffma2_rn(Dyz, dy, __fmul2_rn(Dxz, dx)));
    const float2 q = __ffma2_rn(vz, dz, __ffma2_rn(vy, dy, __fmul2_rn(vx, dx)));       // R.D.R
    const float2 uv = __ffma2_rn(vz, t.uz, __ffma2_rn(vy, t.uy, __fmul2_rn(vx, t.ux)));   // u_k.D.R
    const float2 tr = __fadd2_rn(__fadd2_rn(Dxx, Dyy), Dzz);
    const float2 c1t = __fmul2_rn(c1, tr);
    const float2 e = __ffma2_rn(c2, q, make_float2(-c1t.x, -c1t.y));
    const float2 m2c1 = __fmul2_rn(c1, ff_dup(-2.0f));
    s.hx = __ffma2_rn(e, dx, s.hx); s.hy = __ffma2_rn(e, dy, s.hy); s.hz = __ffma2_rn(e, dz, s.hz);
    s.hx = __ffma2_rn(m2c1, vx, s.hx); s.hy = __ffma2_rn(m2c1, vy, s.hy); s.hz = __ffma2_rn(m2c1, vz, s.hz);
    const float2 c3bq = __fmul2_rn(c3, __fmul2_rn(b, q));
    const float2 gg = __ffma2_rn(c2, __ffma2_rn(ff_dup(2.0f), uv, __fmul2_rn(tr, b)), make_float2(-c3bq.x, -c3bq.y));
    const float2 c2b2 = __fmul2_rn(__fmul2_rn(c2, b), ff_dup(2.0f));
    s.fx = __ffma2_rn(gg, dx, s.fx); s.fy = __ffma2_rn(gg, dy, s.fy); s.fz = __ffma2_rn(gg, dz, s.fz);
    s.fx = __ffma2_rn(c2b2, vx, s.fx); s.fy = __ffma2_rn(c2b2, vy, s.fy); s.fz = __ffma2_rn(c2b2, vz, s.fz);
    s.sk = __fadd2_rn(s.sk, e);
    sq.gxx = __ffma2_rn(c1, Dxx, sq.gxx); sq.gyy = __ffma2_rn(c1, Dyy, sq.gyy); sq.gzz = __ffma2_rn(c1, Dzz, sq.gzz);
    sq.gxy = __ffma2_rn(c1, Dxy, sq.gxy); sq.gxz = __ffma2_rn(c1, Dxz, sq.gxz); sq.gyz = __ffma2_rn(c1, Dyz, sq.gyz);
}
