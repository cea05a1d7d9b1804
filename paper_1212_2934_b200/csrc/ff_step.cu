// ff_step.cu -- the steps either side of the hot path: Lennard-Jones
// short-range force (Eq. 13) and the Euler-Maruyama update
// of the reduced equations of motion Eq. 7-9, i.e. the second half of
// the paper's kernel 5 and its kernel 6.
//
// Rotation is integrated in the vector form of DESIGN.md (reading Q12):
//   d(omega)/dtau = 5/2 (u x h - Gamma_r omega) + noise,   du/dtau = omega x u,  |u| = 1
// which is Eq. 7-8 (2/5 = I / (M R^2)) without the polar-angle singularity.
#include "ff_internal.cuh"

#define FF_LJ_MAX_LEVEL 7                       // cell table of at most 8^7 cells

__device__ __forceinline__ uint32_t ff_compact10(uint32_t v)    // inverse of the 3-way bit spread
{
    v &= 0x09249249u;
    v = (v | (v >> 2)) & 0x030C30C3u;
    v = (v | (v >> 4)) & 0x0300F00Fu;
    v = (v | (v >> 8)) & 0x030000FFu;
    v = (v | (v >> 16)) & 0x000003FFu;
    return v;
}
__device__ __forceinline__ uint32_t ff_spread10s(uint32_t v)
{
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

// deepest level (<= FF_LJ_MAX_LEVEL) whose cell side S 2^-l is still >= the cut-off: computed on the
// device from the device-resident root cube so that ff_step needs no host read
__device__ __forceinline__ int ff_lj_level(float S, float rc)
{
    int lev = 0;
    while (lev < FF_LJ_MAX_LEVEL && ldexpf(S, -(lev + 1)) >= rc) ++lev;
    return lev;
}

// cell table over the level-`lev` cells of the sorted keys: [start, end) per cell prefix
__global__ void __launch_bounds__(256) ff_k_cell_table(const uint32_t* __restrict__ key, int n,
                                                       const ff_globals* __restrict__ g, float rc,
                                                       int32_t* __restrict__ start, int32_t* __restrict__ end)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int lev = ff_lj_level(g->S, rc);
    int sh = 3 * (FF_MAX_LEVEL - lev);
    uint32_t c = __ldg(key + i) >> sh;
    if (i == 0 || (__ldg(key + i - 1) >> sh) != c) start[c] = i;
    if (i == n - 1 || (__ldg(key + i + 1) >> sh) != c) end[c] = i + 1;
}

// Eq. 13: f_k^sr = 24 eps sum_j rho_kj / rho_kj^2 [ (sigma/rho_kj)^12 - (sigma/rho_kj)^6 ], pairs within rc
__global__ void __launch_bounds__(128)
ff_k_lj(const uint32_t* __restrict__ key, const float4* __restrict__ pos_s, const uint32_t* __restrict__ perm, int n,
        const ff_globals* __restrict__ g, const int32_t* __restrict__ start, const int32_t* __restrict__ end, float eps,
        float sigma, float rc, float* __restrict__ fsr)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    int lev = ff_lj_level(g->S, rc);
    float4 p = pos_s[s];
    uint32_t c = __ldg(key + s) >> (3 * (FF_MAX_LEVEL - lev));
    int qx = (int)ff_compact10(c >> 2), qy = (int)ff_compact10(c >> 1), qz = (int)ff_compact10(c);
    const int side = 1 << lev;
    float fx = 0.f, fy = 0.f, fz = 0.f;
    const float rc2 = rc * rc, s2 = sigma * sigma, e24 = 24.0f * eps;
    // Morton codes of the three neighbouring coordinates per axis (0xffffffff = outside the root cube)
    uint32_t mx[3], my[3], mz[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        int x = qx + d - 1, y = qy + d - 1, z = qz + d - 1;
        mx[d] = (x < 0 || x >= side) ? 0xffffffffu : ff_spread10s((uint32_t)x) << 2;
        my[d] = (y < 0 || y >= side) ? 0xffffffffu : ff_spread10s((uint32_t)y) << 1;
        mz[d] = (z < 0 || z >= side) ? 0xffffffffu : ff_spread10s((uint32_t)z);
    }
    // nine (x, y) columns; the table entries of a column's three cells are fetched together, so that a
    // thread exposes 9 table latencies instead of 27
#pragma unroll
    for (int xy = 0; xy < 9; ++xy) {
        const uint32_t cxy = mx[xy / 3] | my[xy % 3];
        if (mx[xy / 3] == 0xffffffffu || my[xy % 3] == 0xffffffffu) continue;
        int b[3], e[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const bool in = mz[d] != 0xffffffffu;
            b[d] = in ? __ldg(start + (cxy | mz[d])) : 0;
            e[d] = in ? __ldg(end + (cxy | mz[d])) : 0;
        }
#pragma unroll
        for (int d = 0; d < 3; ++d)
            for (int j = b[d]; j < e[d]; ++j) {
                FF_CHECK(const_cast<ff_globals*>(g), j >= 0 && j < n);
                const float4 q = __ldg(pos_s + j);
                const float rx = p.x - q.x, ry = p.y - q.y, rz = p.z - q.z;
                const float r2 = fmaf(rz, rz, fmaf(ry, ry, rx * rx));
                if (r2 < rc2 && j != s) {
                    const float ir2 = 1.0f / r2;
                    const float sr2 = s2 * ir2, sr6 = sr2 * sr2 * sr2;
                    const float w = e24 * ir2 * (sr6 * sr6 - sr6);
                    fx = fmaf(w, rx, fx); fy = fmaf(w, ry, fy); fz = fmaf(w, rz, fz);
                }
            }
    }
    size_t o = (size_t)__ldg(perm + s) * 3;
    fsr[o] = fx; fsr[o + 1] = fy; fsr[o + 2] = fz;
}

// counter-based unit Gaussians: splitmix64 finaliser -> Box-Muller
__device__ __forceinline__ uint64_t ff_mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
__device__ __forceinline__ void ff_gauss2(uint64_t seed, uint64_t step, uint64_t k, uint32_t lane, float& g0, float& g1)
{
    uint64_t z = ff_mix64(seed * 0x9E3779B97F4A7C15ull + step);
    z = ff_mix64(z ^ (k * 0xD1B54A32D192ED03ull + lane));
    float u1 = ((float)(uint32_t)(z >> 40) + 0.5f) * (1.0f / 16777216.0f);
    float u2 = ((float)(uint32_t)((z >> 8) & 0xffffffu)) * (1.0f / 16777216.0f);
    float r = sqrtf(-2.0f * __logf(u1));
    __sincosf(6.28318530718f * u2, &g1, &g0);
    g0 *= r; g1 *= r;
}

__global__ void __launch_bounds__(256)
ff_k_integrate(int n, float* __restrict__ pos, float* __restrict__ vel, float* __restrict__ mom,
               float* __restrict__ angvel, const float* __restrict__ H, const float* __restrict__ F,
               const float* __restrict__ fsr, ff_step_params p, uint64_t step)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    size_t o = 3 * (size_t)k;
    float x[3], v[3], u[3], w[3], h[3], f[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        x[a] = pos[o + a]; v[a] = vel[o + a]; u[a] = mom[o + a]; w[a] = angvel[o + a];
        h[a] = H[o + a] + p.h_ext[a];
        f[a] = F[o + a] + (fsr ? fsr[o + a] : 0.0f);
    }
    if (p.wall_epsilon != 0.0f) {
        // container walls (reading Q20): Eq. 13's pair term at the distance to each plane
        const float s2 = p.wall_sigma * p.wall_sigma, e24 = 24.0f * p.wall_epsilon;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const float d0 = x[a] - p.wall_lo[a], d1 = p.wall_hi[a] - x[a];
            if (d0 < p.lj_cutoff) { float i2 = 1.0f / (d0 * d0), s6 = s2 * i2; s6 = s6 * s6 * s6; f[a] += e24 * (s6 * s6 - s6) / d0; }
            if (d1 < p.lj_cutoff) { float i2 = 1.0f / (d1 * d1), s6 = s2 * i2; s6 = s6 * s6 * s6; f[a] -= e24 * (s6 * s6 - s6) / d1; }
        }
    }
    float xi[6] = { 0.f, 0.f, 0.f, 0.f, 0.f, 0.f };
    if (p.noise_d != 0.0f || p.noise_r != 0.0f) {
        ff_gauss2(p.seed, step, (uint64_t)k, 0u, xi[0], xi[1]);
        ff_gauss2(p.seed, step, (uint64_t)k, 1u, xi[2], xi[3]);
        ff_gauss2(p.seed, step, (uint64_t)k, 2u, xi[4], xi[5]);
    }
    float sq = sqrtf(p.dtau);
    // torque u x h
    float t[3] = { u[1] * h[2] - u[2] * h[1], u[2] * h[0] - u[0] * h[2], u[0] * h[1] - u[1] * h[0] };
    // omega x u with the OLD omega (explicit Euler-Maruyama)
    float du[3] = { w[1] * u[2] - w[2] * u[1], w[2] * u[0] - w[0] * u[2], w[0] * u[1] - w[1] * u[0] };
    float un[3], nn = 0.f;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float xn = x[a] + p.dtau * v[a];
        float vn = v[a] + p.dtau * (f[a] - p.gamma_d * v[a]) + p.noise_d * sq * xi[a];
        float wn = w[a] + p.dtau * 2.5f * (t[a] - p.gamma_r * w[a]) + p.noise_r * sq * xi[3 + a];
        un[a] = u[a] + p.dtau * du[a];
        nn += un[a] * un[a];
        pos[o + a] = xn; vel[o + a] = vn; angvel[o + a] = wn;
    }
    float inv = rsqrtf(nn);
#pragma unroll
    for (int a = 0; a < 3; ++a) mom[o + a] = un[a] * inv;
}

// Eq. 13 over the pairs within the cut-off -> c->step_fsr, enqueued on `stream`.  Reads the sorted keys and positions
// of the current tree only.
int ff_launch_lj(ff_ctx* c, int64_t n64, const ff_step_params* p, cudaStream_t stream)
{
    const int n = (int)n64;
    if (!(p->lj_cutoff > 0.0f) || !(p->lj_sigma > 0.0f)) return FF_ERR_INVALID_ARG;
    const size_t cells = (size_t)1 << (3 * FF_LJ_MAX_LEVEL);                // table sized for the deepest level
    int32_t* start = reinterpret_cast<int32_t*>(c->direct_part);          // 2 * 8^7 * 4 B = 16 MB <= scratch
    int32_t* end = start + cells;
    const cudaStream_t main_stream = c->stream;
    c->stream = stream;                                                    // FF_LAUNCH enqueues on c->stream
    int rc = FF_OK;
    auto enqueue = [&]() -> int {
        FF_CUDA(c, cudaMemsetAsync(start, 0, 2 * cells * sizeof(int32_t), c->stream));
        FF_LAUNCH(c, ff_k_cell_table, (n + 255) / 256, 256, 0, c->key[0], n, c->g, p->lj_cutoff, start, end);
        FF_LAUNCH(c, ff_k_lj, (n + 127) / 128, 128, 0, c->key[0], c->pos_s, c->idx[0], n, c->g, start, end,
                  p->lj_epsilon, p->lj_sigma, p->lj_cutoff, c->step_fsr);
        return FF_OK;
    };
    rc = enqueue();
    c->stream = main_stream;
    return rc;
}

int ff_launch_integrate(ff_ctx* c, float* pos, float* vel, float* mom, float* angvel, int64_t n64,
                        const ff_step_params* p, uint64_t step_index, bool with_fsr)
{
    const int n = (int)n64;
    if (p->wall_epsilon != 0.0f && (!(p->lj_cutoff > 0.0f) || !(p->wall_sigma > 0.0f))) return FF_ERR_INVALID_ARG;
    FF_LAUNCH(c, ff_k_integrate, (n + 255) / 256, 256, 0, n, pos, vel, mom, angvel, c->stage_H, c->stage_F,
              with_fsr ? c->step_fsr : (const float*)nullptr, *p, step_index);
    return FF_OK;
}
