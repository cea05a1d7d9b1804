// ff_direct.cu -- a8 tiled all-pairs field + force, and the FP32 FMA-pipe microbenchmark.
//
// Paper: Algorithm 1: one thread per target k, sources staged
// through shared memory in tiles of blockDim.x, self excluded by index (line 5).
// Kept from that design: the tiling and the one-thread-one-target mapping.
// Changed: the self test runs only in the one tile that can contain k (block
// uniform branch); each tile's fp32 partial sums are folded into fp64 running
// sums so that 10^6 sources keep 1e-5 relative accuracy; small N is split over
// source chunks so the grid still covers all 148 SMs.
#include "ff_internal.cuh"
#include "ff_pair.cuh"

// MUFU.RSQ as it is (about 1 ulp): a Newton step was measured to change nothing in the result's error
// (2.9e-6 / 5.4e-6 / 7.9e-6 with and without it on configs 1, 2, 4 against the 1e-5 tolerance), the error
// of a sum is set by the roundings of its 40 other operations per term.
__device__ __forceinline__ float2 ff_rsqrt2(float2 r2) { return make_float2(ff_rsqrt(r2.x), ff_rsqrt(r2.y)); }

#define FF_DIRECT_PAIRS (FF_DIRECT_THREADS / 2)

// grid = (target blocks, source splits).  Block (bx, by) accumulates, for its 256 targets, the
// sources of tiles by, by + splits, by + 2 splits, ...  A tile is staged in shared memory in the pair
// layout of ff_pair.cuh, so that one lane evaluates two sources per packed instruction.
#ifndef FF_DIRECT_MINB
#define FF_DIRECT_MINB 2      // lets ptxas use 92 registers (2 x 8 warps per SM): measured 3 % faster than 66 or 64
#endif
// Lennard-Jones coefficient of Eq. 13 for two sources: w = 24 eps [ (s/r)^12 - (s/r)^6 ] / r^2 inside the cut-off,
// 0 outside and for a masked term (rinv = 0)
struct ff_lj { float e24, s2, rc2; };
__device__ __forceinline__ float2 ff_lj2(float2 r2, float2 rinv, const ff_lj& lj)
{
    const float2 i2 = __fmul2_rn(rinv, rinv);
    const float2 sr2 = __fmul2_rn(i2, ff_dup(lj.s2));
    const float2 sr6 = __fmul2_rn(__fmul2_rn(sr2, sr2), sr2);
    const float2 t = __ffma2_rn(sr6, sr6, make_float2(-sr6.x, -sr6.y));
    const float2 w = __fmul2_rn(t, __fmul2_rn(i2, ff_dup(lj.e24)));
    return make_float2(r2.x < lj.rc2 ? w.x : 0.0f, r2.y < lj.rc2 ? w.y : 0.0f);
}

// LJ = true: the all-pairs MD step of the paper (Algorithm 1 sums f^dip, f^sr and h^dip in one loop): F_out gets
// f^dip + f^sr.
template <bool LJ>
__global__ void __launch_bounds__(FF_DIRECT_THREADS, FF_DIRECT_MINB)
ff_k_direct(const float* __restrict__ pos, const float* __restrict__ mom, int n, int splits,
            double* __restrict__ part, float* __restrict__ H_out, float* __restrict__ F_out, ff_lj lj)
{
    __shared__ float4 tile_q[FF_DIRECT_PAIRS * 3];
    const int t = threadIdx.x;
    const int k = blockIdx.x * FF_DIRECT_THREADS + t;
    const int kk = min(k, n - 1);
    const float ux = __ldg(mom + 3 * (size_t)kk), uy = __ldg(mom + 3 * (size_t)kk + 1), uz = __ldg(mom + 3 * (size_t)kk + 2);
    ff_target2 tg;
    tg.px = ff_dup(__ldg(pos + 3 * (size_t)kk)); tg.py = ff_dup(__ldg(pos + 3 * (size_t)kk + 1));
    tg.pz = ff_dup(__ldg(pos + 3 * (size_t)kk + 2));
    tg.ux = ff_dup(ux); tg.uy = ff_dup(uy); tg.uz = ff_dup(uz);
    double acc[7] = { 0, 0, 0, 0, 0, 0, 0 };
    const int n_tiles = (n + FF_DIRECT_THREADS - 1) / FF_DIRECT_THREADS;
    float* mine = reinterpret_cast<float*>(tile_q) + (t >> 1) * 12 + (t & 1);
    for (int tile = blockIdx.y; tile < n_tiles; tile += splits) {
        int j = tile * FF_DIRECT_THREADS + t;
        float sx = 3.0e18f, sy = 3.0e18f, sz = 3.0e18f, vx = 0.f, vy = 0.f, vz = 0.f;   // padding: zero moment, far away
        if (j < n) {
            sx = __ldg(pos + 3 * (size_t)j); sy = __ldg(pos + 3 * (size_t)j + 1); sz = __ldg(pos + 3 * (size_t)j + 2);
            vx = __ldg(mom + 3 * (size_t)j); vy = __ldg(mom + 3 * (size_t)j + 1); vz = __ldg(mom + 3 * (size_t)j + 2);
        }
        __syncthreads();
        mine[0] = sx; mine[2] = sy; mine[4] = sz; mine[6] = vx; mine[8] = vy; mine[10] = vz;
        __syncthreads();
        // fp32 partial sums over chunks of 32 sources, folded into the fp64 running sums: keeps the
        // accumulation error at sqrt(32) ulp of a chunk sum instead of sqrt(N) ulp of the total
        const bool own = tile == blockIdx.x;     // the only tile that holds this block's own targets
        for (int c0 = 0; c0 < FF_DIRECT_PAIRS; c0 += 16) {
            ff_acc2 s;
            s.hx = s.hy = s.hz = s.fx = s.fy = s.fz = s.sk = ff_dup(0.0f);
            const float4* q = tile_q + 3 * c0;
            if (own) {
#pragma unroll 2
                for (int i = 0; i < 16; ++i) {
                    const float4 q0 = q[3 * i], q1 = q[3 * i + 1], q2 = q[3 * i + 2];
                    float2 dx, dy, dz, r2;
                    ff_pair2_geom(q0, q1, tg, dx, dy, dz, r2);
                    float2 rinv = ff_rsqrt2(r2);
                    if (2 * (c0 + i) == t) rinv.x = 0.0f;          // j != k (Alg. 1 line 5): r2 = 0 gave NaN, dropped here
                    if (2 * (c0 + i) + 1 == t) rinv.y = 0.0f;
                    if (LJ) ff_pair2_accum<true>(q1, q2, tg, dx, dy, dz, rinv, s, ff_lj2(r2, rinv, lj));
                    else ff_pair2_accum(q1, q2, tg, dx, dy, dz, rinv, s);
                }
            } else {
#pragma unroll 4
                for (int i = 0; i < 16; ++i) {
                    const float4 q0 = q[3 * i], q1 = q[3 * i + 1], q2 = q[3 * i + 2];
                    float2 dx, dy, dz, r2;
                    ff_pair2_geom(q0, q1, tg, dx, dy, dz, r2);
                    const float2 rinv = ff_rsqrt2(r2);
                    if (LJ) ff_pair2_accum<true>(q1, q2, tg, dx, dy, dz, rinv, s, ff_lj2(r2, rinv, lj));
                    else ff_pair2_accum(q1, q2, tg, dx, dy, dz, rinv, s);
                }
            }
            acc[0] += s.hx.x + s.hx.y; acc[1] += s.hy.x + s.hy.y; acc[2] += s.hz.x + s.hz.y;
            acc[3] += s.fx.x + s.fx.y; acc[4] += s.fy.x + s.fy.y; acc[5] += s.fz.x + s.fz.y;
            acc[6] += s.sk.x + s.sk.y;
        }
    }
    if (k >= n) return;
    acc[3] += acc[6] * (double)ux; acc[4] += acc[6] * (double)uy; acc[5] += acc[6] * (double)uz;
    if (splits == 1) {
        if (H_out) { H_out[3 * (size_t)k] = (float)acc[0]; H_out[3 * (size_t)k + 1] = (float)acc[1]; H_out[3 * (size_t)k + 2] = (float)acc[2]; }
        if (F_out) { F_out[3 * (size_t)k] = (float)acc[3]; F_out[3 * (size_t)k + 1] = (float)acc[4]; F_out[3 * (size_t)k + 2] = (float)acc[5]; }
    } else {
        double* p = part + ((size_t)blockIdx.y * n + k) * 6;
#pragma unroll
        for (int a = 0; a < 6; ++a) p[a] = acc[a];
    }
}

__global__ void __launch_bounds__(256)
ff_k_direct_reduce(const double* __restrict__ part, int n, int splits, float* __restrict__ H_out, float* __restrict__ F_out)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    double acc[6] = { 0, 0, 0, 0, 0, 0 };
    for (int s = 0; s < splits; ++s) {
        const double* p = part + ((size_t)s * n + k) * 6;
#pragma unroll
        for (int a = 0; a < 6; ++a) acc[a] += p[a];
    }
    if (H_out) { H_out[3 * (size_t)k] = (float)acc[0]; H_out[3 * (size_t)k + 1] = (float)acc[1]; H_out[3 * (size_t)k + 2] = (float)acc[2]; }
    if (F_out) { F_out[3 * (size_t)k] = (float)acc[3]; F_out[3 * (size_t)k + 1] = (float)acc[4]; F_out[3 * (size_t)k + 2] = (float)acc[5]; }
}

int ff_launch_direct(ff_ctx* c, const float* pos, const float* mom, int64_t n64, float* H_out, float* F_out,
                     float lj_eps, float lj_sigma, float lj_cutoff)
{
    int n = (int)n64;
    int tblocks = (n + FF_DIRECT_THREADS - 1) / FF_DIRECT_THREADS;
    // enough blocks for ~4 per SM; the partial-sum scratch bounds targets * splits
    int want = c->num_sms * 4;
    int splits = (want + tblocks - 1) / tblocks;
    if (splits > tblocks) splits = tblocks;
    while (splits > 1 && (int64_t)splits * n > FF_DIRECT_SPLIT_ELEMS) --splits;
    if (splits < 1) splits = 1;
    dim3 grid(tblocks, splits);
    ff_lj lj = { 24.0f * lj_eps, lj_sigma * lj_sigma, lj_cutoff * lj_cutoff };
    if (lj_eps != 0.0f)
        FF_LAUNCH(c, ff_k_direct<true>, grid, FF_DIRECT_THREADS, 0, pos, mom, n, splits, c->direct_part, H_out, F_out, lj);
    else
        FF_LAUNCH(c, ff_k_direct<false>, grid, FF_DIRECT_THREADS, 0, pos, mom, n, splits, c->direct_part, H_out, F_out, lj);
    if (splits > 1)
        FF_LAUNCH(c, ff_k_direct_reduce, (n + 255) / 256, 256, 0, c->direct_part, n, splits, H_out, F_out);
    return FF_OK;
}

// ---- FP32 FMA-pipe peak: 8 independent dependent chains per thread ---------------------
__global__ void __launch_bounds__(256) ff_k_fma_peak(int iters, float seed, float* __restrict__ sink)
{
    float x0 = seed + threadIdx.x, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f,
          x6 = x0 + 6.f, x7 = x0 + 7.f;
    const float a = 0.999f + seed * 1e-9f, b = 1e-3f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
            x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
        }
    }
    float s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 12345.678f) sink[0] = s;          // never true in practice; keeps the chains alive
}

int ff_launch_fp32_peak(ff_ctx* c, int iters, double* tflops)
{
    if (iters < 1) iters = 1;
    int blocks = c->num_sms * 8;
    cudaEvent_t e0, e1;
    FF_CUDA(c, cudaEventCreate(&e0));
    FF_CUDA(c, cudaEventCreate(&e1));
    float* sink = reinterpret_cast<float*>(c->direct_part);
    FF_LAUNCH(c, ff_k_fma_peak, blocks, 256, 0, iters, 1.0f, sink);     // warm-up
    FF_CUDA(c, cudaEventRecord(e0, c->stream));
    FF_LAUNCH(c, ff_k_fma_peak, blocks, 256, 0, iters, 1.0f, sink);
    FF_CUDA(c, cudaEventRecord(e1, c->stream));
    FF_CUDA(c, cudaEventSynchronize(e1));
    float ms = 0.f;
    FF_CUDA(c, cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    double flop = 2.0 * 64.0 * (double)iters * 256.0 * (double)blocks;
    *tflops = flop / ((double)ms * 1e-3) / 1e12;
    return FF_OK;
}
