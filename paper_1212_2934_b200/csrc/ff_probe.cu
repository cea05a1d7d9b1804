// ff_probe.cu -- FP32-pipe probes: what the ALU roofline of the walk and of the direct kernel is measured against.
//
// MEASURED_PEAKS.json holds no FP32 figure, so bench.py measures one in the same run.  The nominal
// peak (SMs x 128 lanes x 2 flop x clock) is reached only by FMAs whose operands do not all come from the register
// file: the register file delivers one even and one odd 32-bit register per lane and cycle, so a packed FFMA2 with
// three register-PAIR operands issues every 3 cycles instead of every 2, and one with a reused (or immediate, or
// scalar-broadcast) operand every 2 to 2.5.  The probes time exactly those forms and the evaluation loop of the walk
// by itself (ff_pair.cuh on a shared-memory batch), which is the ceiling of ff_k_walk and ff_k_direct.
#include "ff_internal.cuh"
#include "ff_pair.cuh"

#define FF_PROBE_THREADS 256
#define FF_PROBE_CHAINS 8

// kind 0: scalar FFMA x = x * a + b, a and b shared by the 8 chains (they sit in the operand reuse cache)
__global__ void __launch_bounds__(FF_PROBE_THREADS) ff_k_probe_ffma(int iters, float seed, float* __restrict__ sink)
{
    float x[FF_PROBE_CHAINS];
#pragma unroll
    for (int c = 0; c < FF_PROBE_CHAINS; ++c) x[c] = seed + threadIdx.x + c;
    const float a = 0.999f + seed * 1e-9f, b = 1e-3f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int c = 0; c < FF_PROBE_CHAINS; ++c) x[c] = fmaf(x[c], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < FF_PROBE_CHAINS; ++c) s += x[c];
    if (s == 12345.678f) sink[0] = s;          // never true in practice; keeps the chains alive
}

// kinds 1-3: packed FFMA2 x_c = y_c * z_c + x_c with 8 independent chains
//   FORM 1  y_c, z_c distinct register pairs per chain           (three register-pair operands)
//   FORM 2  y shared by all chains, z_c distinct                 (one operand served by the reuse cache)
//   FORM 3  y a scalar in the broadcast operand form, z_c pairs  (the form the evaluation loop uses for sources)
template <int FORM>
__global__ void __launch_bounds__(FF_PROBE_THREADS) ff_k_probe_ffma2(int iters, float seed, float* __restrict__ sink)
{
    float2 x[FF_PROBE_CHAINS], y[FF_PROBE_CHAINS], z[FF_PROBE_CHAINS];
#pragma unroll
    for (int c = 0; c < FF_PROBE_CHAINS; ++c) {
        x[c] = make_float2(seed + threadIdx.x + c, seed - c);
        y[c] = make_float2(0.999f + 1e-6f * (threadIdx.x + c), 0.998f + 1e-6f * c);
        z[c] = make_float2(1.0f - 1e-6f * (threadIdx.x + 2 * c), 1.0f + 1e-6f * c);
    }
    const float ys = 0.999f + seed * 1e-9f + 1e-7f * threadIdx.x;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int c = 0; c < FF_PROBE_CHAINS; ++c) {
                if (FORM == 1) x[c] = __ffma2_rn(y[c], z[c], x[c]);
                else if (FORM == 2) x[c] = __ffma2_rn(y[0], z[c], x[c]);
                else x[c] = __ffma2_rn(ff_dup(ys), z[c], x[c]);
            }
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < FF_PROBE_CHAINS; ++c) s += x[c].x + x[c].y;
    if (s == 12345.678f) sink[0] = s;
}

// kind 4: the evaluation loop of the walk alone -- every lane evaluates a batch of 32 shared-memory source records
// for its two targets exactly as ff_k_walk<32> does (half-warps take the even / odd records), over and over.
// Launched with the walk's block shape and residency (4 warps per block, FF_WALK_MINB blocks per SM).
// MODE 0: the loop as the kernels have it (ff_pair2g: 36 packed instructions).  MODE 1: the same 36 operations per target
// written on scalars (72 FFMA / FMUL per source and pair of targets, no packed instruction).  MODE 2: packed wherever
// an operand is a broadcast scalar or repeats, but the twelve FFMA2 whose three operands are three different register
// pairs (h += (p rho) a, T += (p rho) e, G += (p rho) e: 3 + 3 + 6) as 24 scalar FFMA.  Modes 1 and 2 answer whether the
// packed form's operand bandwidth or the arithmetic itself bounds the loop.
struct ff_probe_acc1 { float hx, hy, hz, txx, tyy, tzz, gxy, gxz, gyz; };

__device__ __forceinline__ void ff_probe_pair1(const float4& A, const float2& B, float px_, float py_, float pz_,
                                               ff_probe_acc1& s)
{
    const float dx = px_ - A.x, dy = py_ - A.y, dz = pz_ - A.z;
    const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
    const float rinv = ff_rsqrt(r2);
    const float mx = A.w, my = B.x, mz = B.y;
    const float rinv2 = __fmul_rn(rinv, rinv);
    const float nr3 = __fmul_rn(rinv2, -rinv);
    const float p = __fmul_rn(nr3, __fmul_rn(rinv2, -3.0f));
    const float a = __fmaf_rn(mz, dz, __fmaf_rn(my, dy, __fmul_rn(mx, dx)));
    const float px = __fmul_rn(p, dx), py = __fmul_rn(p, dy), pz = __fmul_rn(p, dz);
    s.hx = __fmaf_rn(px, a, s.hx); s.hy = __fmaf_rn(py, a, s.hy); s.hz = __fmaf_rn(pz, a, s.hz);
    s.hx = __fmaf_rn(nr3, mx, s.hx); s.hy = __fmaf_rn(nr3, my, s.hy); s.hz = __fmaf_rn(nr3, mz, s.hz);
    const float m = __fmul_rn(a, __fmul_rn(rinv2, -2.5f));
    const float ex = __fmaf_rn(m, dx, mx), ey = __fmaf_rn(m, dy, my), ez = __fmaf_rn(m, dz, mz);
    s.txx = __fmaf_rn(px, ex, s.txx); s.tyy = __fmaf_rn(py, ey, s.tyy); s.tzz = __fmaf_rn(pz, ez, s.tzz);
    s.gxy = __fmaf_rn(px, ey, s.gxy); s.gxy = __fmaf_rn(py, ex, s.gxy);
    s.gxz = __fmaf_rn(px, ez, s.gxz); s.gxz = __fmaf_rn(pz, ex, s.gxz);
    s.gyz = __fmaf_rn(py, ez, s.gyz); s.gyz = __fmaf_rn(pz, ey, s.gyz);
}

#define FF_S2(acc, u, v) do { acc.x = __fmaf_rn(u.x, v.x, acc.x); acc.y = __fmaf_rn(u.y, v.y, acc.y); } while (0)
__device__ __forceinline__ void ff_probe_pair2_hybrid(const float4& A, const float2& B, const ff_target2& t, ff_accg2& s)
{
    float2 dx, dy, dz, r2;
    ff_pair2_geom(A, t, dx, dy, dz, r2);
    const float2 rinv = ff_rsqrt2(r2);
    const float2 mx = ff_dup(A.w), my = ff_dup(B.x), mz = ff_dup(B.y);
    const float2 rinv2 = __fmul2_rn(rinv, rinv);
    const float2 nr3 = __fmul2_rn(rinv2, make_float2(-rinv.x, -rinv.y));
    const float2 p = __fmul2_rn(nr3, __fmul2_rn(rinv2, ff_dup(-3.0f)));
    const float2 a = __ffma2_rn(mz, dz, __ffma2_rn(my, dy, __fmul2_rn(mx, dx)));
    const float2 px = __fmul2_rn(p, dx), py = __fmul2_rn(p, dy), pz = __fmul2_rn(p, dz);
    FF_S2(s.hx, px, a); FF_S2(s.hy, py, a); FF_S2(s.hz, pz, a);
    s.hx = __ffma2_rn(nr3, mx, s.hx); s.hy = __ffma2_rn(nr3, my, s.hy); s.hz = __ffma2_rn(nr3, mz, s.hz);
    const float2 m = __fmul2_rn(a, __fmul2_rn(rinv2, ff_dup(-2.5f)));
    const float2 ex = __ffma2_rn(m, dx, mx), ey = __ffma2_rn(m, dy, my), ez = __ffma2_rn(m, dz, mz);
    FF_S2(s.txx, px, ex); FF_S2(s.tyy, py, ey); FF_S2(s.tzz, pz, ez);
    FF_S2(s.gxy, px, ey); FF_S2(s.gxy, py, ex);
    FF_S2(s.gxz, px, ez); FF_S2(s.gxz, pz, ex);
    FF_S2(s.gyz, py, ez); FF_S2(s.gyz, pz, ey);
}
#undef FF_S2

template <int MODE>
__global__ void __launch_bounds__(FF_WALK_WARPS * 32, FF_WALK_MINB)
ff_k_probe_eval(int iters, float seed, float* __restrict__ sink)
{
    __shared__ float4 qa[FF_WALK_WARPS][32];
    __shared__ float2 qb[FF_WALK_WARPS][32];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31, half = lane >> 4;
    qa[w][lane] = make_float4(100.f + lane + seed, 200.f + 2.f * lane, 50.f - lane, 0.3f + 0.01f * lane);
    qb[w][lane] = make_float2(0.5f - 0.01f * lane, 0.8f);
    __syncwarp();
    ff_target2 tg;
    const float b = (lane & 15) * 0.37f + blockIdx.x * 1e-3f;
    tg.px = make_float2(b, b + 6.f); tg.py = make_float2(b * 0.5f + 1.f, b * 0.5f + 4.f); tg.pz = make_float2(2.f - b, -4.f - b);
    tg.ux = make_float2(0.6f + 1e-3f * lane, 0.8f - 1e-3f * lane); tg.uy = make_float2(1e-3f * lane, -1e-3f * lane);
    tg.uz = make_float2(0.8f, 0.6f);
    ff_accg2 s;
    ff_accg2_zero(s);
    ff_probe_acc1 s0 = { 0, 0, 0, 0, 0, 0, 0, 0, 0 }, s1 = s0;
    for (int it = 0; it < iters; ++it) {
        const float4* pa = qa[w] + half;
        const float2* pb = qb[w] + half;
#pragma unroll 4
        for (int i = 0; i < 16; ++i) {
            if (MODE == 0) ff_pair2g(pa[2 * i], pb[2 * i], tg, s);
            else if (MODE == 2) ff_probe_pair2_hybrid(pa[2 * i], pb[2 * i], tg, s);
            else {
                const float4 A = pa[2 * i];
                const float2 B = pb[2 * i];
                ff_probe_pair1(A, B, tg.px.x, tg.py.x, tg.pz.x, s0);
                ff_probe_pair1(A, B, tg.px.y, tg.py.y, tg.pz.y, s1);
            }
        }
        __syncwarp();
    }
    float r = s.hx.x + s.hx.y + s.hy.x + s.hy.y + s.hz.x + s.hz.y + s.txx.x + s.txx.y + s.tyy.x + s.tyy.y + s.tzz.x +
              s.tzz.y + s.gxy.x + s.gxy.y + s.gxz.x + s.gxz.y + s.gyz.x + s.gyz.y;
    r += s0.hx + s0.hy + s0.hz + s0.txx + s0.tyy + s0.tzz + s0.gxy + s0.gxz + s0.gyz;
    r += s1.hx + s1.hy + s1.hz + s1.txx + s1.tyy + s1.tzz + s1.gxy + s1.gxz + s1.gyz;
    if (r == 12345.678f) sink[0] = r;
}

template <class K>
static int ff_time_probe(ff_ctx* c, K kernel, int blocks, int threads, int iters, float* sink, float* ms)
{
    cudaEvent_t e0, e1;
    FF_CUDA(c, cudaEventCreate(&e0));
    FF_CUDA(c, cudaEventCreate(&e1));
    FF_LAUNCH(c, kernel, blocks, threads, 0, max(1, iters / 16), 1.0f, sink);      // warm-up
    FF_CUDA(c, cudaEventRecord(e0, c->stream));
    FF_LAUNCH(c, kernel, blocks, threads, 0, iters, 1.0f, sink);
    FF_CUDA(c, cudaEventRecord(e1, c->stream));
    FF_CUDA(c, cudaEventSynchronize(e1));
    FF_CUDA(c, cudaEventElapsedTime(ms, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return FF_OK;
}

int ff_launch_probe(ff_ctx* c, int kind, int iters, double* tflops)
{
    if (iters < 1) iters = 1;
    float* sink = reinterpret_cast<float*>(c->direct_part);
    float ms = 0.f;
    int rc;
    double flop;
    if (kind == FF_PROBE_EVAL || kind == FF_PROBE_EVAL_SCALAR || kind == FF_PROBE_EVAL_HYBRID) {
        void (*kernel)(int, float, float*) = kind == FF_PROBE_EVAL ? ff_k_probe_eval<0>
                                           : kind == FF_PROBE_EVAL_SCALAR ? ff_k_probe_eval<1> : ff_k_probe_eval<2>;
        int per_sm = 0;
        FF_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, FF_WALK_WARPS * 32, 0));
        per_sm = max(1, min(per_sm, FF_WALK_MINB));
        const int blocks = c->num_sms * per_sm;
        if ((rc = ff_time_probe(c, kernel, blocks, FF_WALK_WARPS * 32, iters, sink, &ms)) != FF_OK) return rc;
        // per warp and iteration: 32 records x 32 targets = 1024 interactions of 60 flop
        flop = 60.0 * 1024.0 * (double)iters * FF_WALK_WARPS * (double)blocks;
    } else {
        const int blocks = c->num_sms * 8;
        switch (kind) {
        case FF_PROBE_FFMA: rc = ff_time_probe(c, ff_k_probe_ffma, blocks, FF_PROBE_THREADS, iters, sink, &ms); break;
        case FF_PROBE_FFMA2_PAIRS: rc = ff_time_probe(c, ff_k_probe_ffma2<1>, blocks, FF_PROBE_THREADS, iters, sink, &ms); break;
        case FF_PROBE_FFMA2_REUSE: rc = ff_time_probe(c, ff_k_probe_ffma2<2>, blocks, FF_PROBE_THREADS, iters, sink, &ms); break;
        case FF_PROBE_FFMA2_SCALAR: rc = ff_time_probe(c, ff_k_probe_ffma2<3>, blocks, FF_PROBE_THREADS, iters, sink, &ms); break;
        default: return FF_ERR_INVALID_ARG;
        }
        if (rc != FF_OK) return rc;
        const double lanes = kind == FF_PROBE_FFMA ? 1.0 : 2.0;          // FMAs per thread and instruction
        flop = 2.0 * lanes * 8.0 * FF_PROBE_CHAINS * (double)iters * FF_PROBE_THREADS * (double)blocks;
    }
    *tflops = flop / ((double)ms * 1e-3) / 1e12;
    return FF_OK;
}
