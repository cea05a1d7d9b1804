// ff_direct.cu -- a8 tiled all-pairs field + force.
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

#define FF_DIRECT_TARGETS (2 * FF_DIRECT_THREADS)   // two targets per thread (ff_pair.cuh)

// grid = (target blocks, source splits).  Block (bx, by) accumulates, for its 512 targets (thread t: targets
// 512 bx + t and 512 bx + 256 + t), the sources of tiles by, by + splits, by + 2 splits, ...  A tile of 256 sources
// is staged in shared memory as one 32-byte record per source (x, y, z, mx | my, mz), read by broadcast loads; one
// packed instruction evaluates one source against the thread's two targets.
#ifndef FF_DIRECT_MINB
#define FF_DIRECT_MINB 2
#endif
// Lennard-Jones coefficient of Eq. 13 for one source and two targets: w = 24 eps [ (s/r)^12 - (s/r)^6 ] / r^2 inside
// the cut-off, 0 outside and for a masked term (rinv = 0)
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
    __shared__ float4 tileA[FF_DIRECT_THREADS];
    __shared__ float2 tileB[FF_DIRECT_THREADS];
    const int t = threadIdx.x;
    const int k0 = blockIdx.x * FF_DIRECT_TARGETS + t, k1 = k0 + FF_DIRECT_THREADS;
    const size_t o0 = 3 * (size_t)min(k0, n - 1), o1 = 3 * (size_t)min(k1, n - 1);
    ff_target2 tg;
    tg.px = ff_pin_pair(__ldg(pos + o0), __ldg(pos + o1));
    tg.py = ff_pin_pair(__ldg(pos + o0 + 1), __ldg(pos + o1 + 1));
    tg.pz = ff_pin_pair(__ldg(pos + o0 + 2), __ldg(pos + o1 + 2));
    tg.ux = ff_pin_pair(__ldg(mom + o0), __ldg(mom + o1));
    tg.uy = ff_pin_pair(__ldg(mom + o0 + 1), __ldg(mom + o1 + 1));
    tg.uz = ff_pin_pair(__ldg(mom + o0 + 2), __ldg(mom + o1 + 2));
    // fp64 running sums per target: h (3), T_aa (3), G_ab (3) of the tensor form (ff_pair.cuh), f^sr (3, LJ only)
    double acc0[12] = { 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0 }, acc1[12] = { 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0 };
    const int n_tiles = (n + FF_DIRECT_THREADS - 1) / FF_DIRECT_THREADS;
    for (int tile = blockIdx.y; tile < n_tiles; tile += splits) {
        const int j = tile * FF_DIRECT_THREADS + t;
        float sx = 3.0e18f, sy = 3.0e18f, sz = 3.0e18f, vx = 0.f, vy = 0.f, vz = 0.f;   // padding: zero moment, far away
        if (j < n) {
            sx = __ldg(pos + 3 * (size_t)j); sy = __ldg(pos + 3 * (size_t)j + 1); sz = __ldg(pos + 3 * (size_t)j + 2);
            vx = __ldg(mom + 3 * (size_t)j); vy = __ldg(mom + 3 * (size_t)j + 1); vz = __ldg(mom + 3 * (size_t)j + 2);
        }
        __syncthreads();
        tileA[t] = make_float4(sx, sy, sz, vx);
        tileB[t] = make_float2(vy, vz);
        __syncthreads();
        // fp32 partial sums over chunks of 32 sources, folded into the fp64 running sums: keeps the
        // accumulation error at sqrt(32) ulp of a chunk sum instead of sqrt(N) ulp of the total.
        // Tiles 2 bx and 2 bx + 1 are the only ones that hold this block's own targets (first / second of a thread).
        const bool own = (tile >> 1) == (int)blockIdx.x;
        const bool own_second = tile & 1;
        for (int c0 = 0; c0 < FF_DIRECT_THREADS; c0 += 32) {
            ff_accg2 s;
            ff_accg2_zero(s);
            float2 lx = ff_dup(0.0f), ly = lx, lz = lx;     // LJ: sum_j w rho
            if (own) {
#pragma unroll 2
                for (int i = 0; i < 32; ++i) {
                    const float4 A = tileA[c0 + i];
                    const float2 B = tileB[c0 + i];
                    float2 dx, dy, dz, r2;
                    ff_pair2_geom(A, tg, dx, dy, dz, r2);
                    float2 rinv = ff_rsqrt2(r2);
                    if (c0 + i == t) {                     // j != k (Alg. 1 line 5): r2 = 0 gave inf, dropped here
                        if (own_second) rinv.y = 0.0f; else rinv.x = 0.0f;
                    }
                    ff_pair2g_accum(A, B, dx, dy, dz, rinv, s);
                    if (LJ) {
                        const float2 w = ff_lj2(r2, rinv, lj);
                        lx = __ffma2_rn(w, dx, lx); ly = __ffma2_rn(w, dy, ly); lz = __ffma2_rn(w, dz, lz);
                    }
                }
            } else {
#pragma unroll 4
                for (int i = 0; i < 32; ++i) {
                    const float4 A = tileA[c0 + i];
                    const float2 B = tileB[c0 + i];
                    if (LJ) {
                        float2 dx, dy, dz, r2;
                        ff_pair2_geom(A, tg, dx, dy, dz, r2);
                        const float2 rinv = ff_rsqrt2(r2);
                        ff_pair2g_accum(A, B, dx, dy, dz, rinv, s);
                        const float2 w = ff_lj2(r2, rinv, lj);
                        lx = __ffma2_rn(w, dx, lx); ly = __ffma2_rn(w, dy, ly); lz = __ffma2_rn(w, dz, lz);
                    } else {
                        ff_pair2g(A, B, tg, s);
                    }
                }
            }
            acc0[0] += s.hx.x; acc0[1] += s.hy.x; acc0[2] += s.hz.x; acc0[3] += s.txx.x; acc0[4] += s.tyy.x;
            acc0[5] += s.tzz.x; acc0[6] += s.gxy.x; acc0[7] += s.gxz.x; acc0[8] += s.gyz.x;
            acc1[0] += s.hx.y; acc1[1] += s.hy.y; acc1[2] += s.hz.y; acc1[3] += s.txx.y; acc1[4] += s.tyy.y;
            acc1[5] += s.tzz.y; acc1[6] += s.gxy.y; acc1[7] += s.gxz.y; acc1[8] += s.gyz.y;
            if (LJ) {
                acc0[9] += lx.x; acc0[10] += ly.x; acc0[11] += lz.x;
                acc1[9] += lx.y; acc1[10] += ly.y; acc1[11] += lz.y;
            }
        }
    }
    auto finish = [&](int k, double* acc, float ux, float uy, float uz) {
        if (k >= n) return;
        // f = G u_k (+ f^sr): G_aa = 2 T_aa + S, S = sum_j p a = -(2/3) tr T (the tensor is traceless term by term)
        const double S = -(2.0 / 3.0) * (acc[3] + acc[4] + acc[5]);
        const double gxx = 2.0 * acc[3] + S, gyy = 2.0 * acc[4] + S, gzz = 2.0 * acc[5] + S;
        const double fx = gxx * ux + acc[6] * uy + acc[7] * uz + acc[9];
        const double fy = acc[6] * ux + gyy * uy + acc[8] * uz + acc[10];
        const double fz = acc[7] * ux + acc[8] * uy + gzz * uz + acc[11];
        acc[3] = fx; acc[4] = fy; acc[5] = fz;
        if (splits == 1) {
            if (H_out) { H_out[3 * (size_t)k] = (float)acc[0]; H_out[3 * (size_t)k + 1] = (float)acc[1]; H_out[3 * (size_t)k + 2] = (float)acc[2]; }
            if (F_out) { F_out[3 * (size_t)k] = (float)acc[3]; F_out[3 * (size_t)k + 1] = (float)acc[4]; F_out[3 * (size_t)k + 2] = (float)acc[5]; }
        } else {
            double* p = part + ((size_t)blockIdx.y * n + k) * 6;
#pragma unroll
            for (int a = 0; a < 6; ++a) p[a] = acc[a];
        }
    };
    finish(k0, acc0, tg.ux.x, tg.uy.x, tg.uz.x);
    finish(k1, acc1, tg.ux.y, tg.uy.y, tg.uz.y);
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
    int tblocks = (n + FF_DIRECT_TARGETS - 1) / FF_DIRECT_TARGETS;
    // enough blocks for ~4 per SM; the partial-sum scratch bounds targets * splits
    int want = c->num_sms * 4;
    int splits = (want + tblocks - 1) / tblocks;
    const int n_tiles = (n + FF_DIRECT_THREADS - 1) / FF_DIRECT_THREADS;
    if (splits > n_tiles) splits = n_tiles;
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

// ---- ff_eval_direct_static: the all-pairs sum for callers that cannot allocate (include/ff.h) --------------------
// The split kernel above parks one fp64 partial sum per (source split, target) in scratch before ff_k_direct_reduce
// folds them.  Every other entry point takes that scratch from the caller's workspace; this one takes it from a
// fixed array that is part of the library image, so it needs no context, no workspace and no allocation call.
// The price: every GPU that loads libff.so carries these 3 MiB until the process exits, n is capped at
// FF_STATIC_MAX_N, and all calls share the one array.
#include <mutex>

#define FF_STATIC_PART_ELEMS (2 * FF_STATIC_MAX_N)      // (split, target) pairs the array holds: 65 536 x 48 B = 3 MiB
#define FF_STATIC_MAX_DEVICES 64

static __device__ __align__(256) double ff_static_part[(size_t)FF_STATIC_PART_ELEMS * 6];

namespace {
// In host code `ff_static_part` is only a handle for the runtime, not an address a kernel can use: the device
// address is asked for once per device (with that device current) and kept here.
struct ff_static_dev { double* part; int num_sms; bool ready; };
ff_static_dev ff_static_devs[FF_STATIC_MAX_DEVICES];
std::mutex ff_static_mutex;
thread_local char ff_static_error[256] = "";

int ff_static_fail(int code, const char* what, const char* detail)
{
    snprintf(ff_static_error, sizeof(ff_static_error), "%s: %s", what, detail);
    return code;
}
}   // namespace

extern "C" const char* ff_static_last_error(void) { return ff_static_error; }

extern "C" int ff_eval_direct_static(const float* pos, const float* mom, int64_t n, float* H_out, float* F_out,
                                     void* cuda_stream)
{
    ff_static_error[0] = 0;
    if (!pos || !mom || n <= 0 || (!H_out && !F_out))
        return ff_static_fail(FF_ERR_INVALID_ARG, "ff_eval_direct_static", "NULL pos/mom, n <= 0 or no output array");
    if (n > FF_STATIC_MAX_N) {
        char msg[160];
        snprintf(msg, sizeof(msg), "n = %lld is beyond FF_STATIC_MAX_N = %d, the most the built-in scratch array holds; "
                 "use ff_eval_direct with a workspace", (long long)n, (int)FF_STATIC_MAX_N);
        return ff_static_fail(FF_ERR_TOO_LARGE, "ff_eval_direct_static", msg);
    }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return ff_static_fail(FF_ERR_CUDA, "cudaGetDevice", cudaGetErrorString(e));
    if (dev < 0 || dev >= FF_STATIC_MAX_DEVICES)
        return ff_static_fail(FF_ERR_INVALID_ARG, "ff_eval_direct_static", "device ordinal beyond FF_STATIC_MAX_DEVICES");
    ff_static_dev sd;
    {
        // first call on this device: look the array's device address up (this may load the module's kernels, which
        // is why the first call belongs before any stream capture)
        std::lock_guard<std::mutex> lock(ff_static_mutex);
        ff_static_dev& slot = ff_static_devs[dev];
        if (!slot.ready) {
            double* p = nullptr;
            e = cudaGetSymbolAddress((void**)&p, ff_static_part);
            if (e != cudaSuccess || !p)
                return ff_static_fail(FF_ERR_CUDA, "cudaGetSymbolAddress(ff_static_part)", cudaGetErrorString(e));
            int sms = 0;
            e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            if (e != cudaSuccess || sms <= 0)
                return ff_static_fail(FF_ERR_CUDA, "cudaDeviceGetAttribute(multiProcessorCount)", cudaGetErrorString(e));
            slot.part = p; slot.num_sms = sms; slot.ready = true;
        }
        sd = slot;
    }
    // the grid of ff_launch_direct, with the split count bounded by what the array holds.  Nothing in the array has
    // to start at zero: block (bx, by) overwrites all six sums of each of its (by, k) records, and the reduction
    // reads only records [0, splits) x [0, n), so what an earlier call left behind is never read.
    const int ni = (int)n;
    const int tblocks = (ni + FF_DIRECT_TARGETS - 1) / FF_DIRECT_TARGETS;
    const int n_tiles = (ni + FF_DIRECT_THREADS - 1) / FF_DIRECT_THREADS;
    int splits = (sd.num_sms * 4 + tblocks - 1) / tblocks;
    if (splits > n_tiles) splits = n_tiles;
    if ((int64_t)splits * ni > FF_STATIC_PART_ELEMS) splits = (int)(FF_STATIC_PART_ELEMS / ni);
    if (splits < 1) splits = 1;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const ff_lj lj = { 0.0f, 1.0f, 0.0f };
    ff_k_direct<false><<<dim3(tblocks, splits), FF_DIRECT_THREADS, 0, stream>>>(pos, mom, ni, splits, sd.part, H_out, F_out, lj);
    if ((e = cudaGetLastError()) != cudaSuccess) return ff_static_fail(FF_ERR_CUDA, "ff_k_direct", cudaGetErrorString(e));
    if (splits > 1) {
        ff_k_direct_reduce<<<(ni + 255) / 256, 256, 0, stream>>>(sd.part, ni, splits, H_out, F_out);
        if ((e = cudaGetLastError()) != cudaSuccess)
            return ff_static_fail(FF_ERR_CUDA, "ff_k_direct_reduce", cudaGetErrorString(e));
    }
    return FF_OK;
}
