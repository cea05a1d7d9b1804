// ff_sort.cu -- a1 bounding box, a2 Morton keys, a3 stable LSD radix sort + gather.
//
// Paper: kernel 1 "bounding box" and kernel 4 "sorting of the
// particles with respect to their positions".  Here the sort comes
// FIRST and the octree is derived from the sorted keys (ff_build.cu), which
// replaces the paper's lock-based insertion.
//
// All phases are HBM/L2 streaming work: coalesced loads, no tensor cores.
#include "ff_internal.cuh"

// ------------------------------------------------------------------ a1 bbox --
__global__ void ff_k_reset(ff_globals* g)
{
    int t = threadIdx.x;
    if (t < 3) { g->bbox_ord[t] = 0xffffffffu; g->bbox_ord[4 + t] = 0u; }
    if (t < 4) g->counters[t] = 0ull;
    if (t == 0) { g->n_cells = 0; g->max_level = 0; }
    if (t < FF_MAX_LEVEL) { g->level_count[t] = 0; g->level_cursor[t] = 0; }
}

__global__ void __launch_bounds__(256) ff_k_bbox(const float* __restrict__ pos, int n, ff_globals* g)
{
    uint32_t mn[3] = { 0xffffffffu, 0xffffffffu, 0xffffffffu }, mx[3] = { 0u, 0u, 0u };
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            uint32_t o = ff_f2ord(__ldg(pos + 3 * (size_t)i + a));
            mn[a] = min(mn[a], o);
            mx[a] = max(mx[a], o);
        }
    }
    __shared__ uint32_t smn[3], smx[3];
    if (threadIdx.x < 3) { smn[threadIdx.x] = 0xffffffffu; smx[threadIdx.x] = 0u; }
    __syncthreads();
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        uint32_t lo = __reduce_min_sync(FF_FULL, mn[a]);
        uint32_t hi = __reduce_max_sync(FF_FULL, mx[a]);
        if (ff_lane() == 0) { atomicMin(&smn[a], lo); atomicMax(&smx[a], hi); }
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        atomicMin(&g->bbox_ord[threadIdx.x], smn[threadIdx.x]);
        atomicMax(&g->bbox_ord[4 + threadIdx.x], smx[threadIdx.x]);
    }
}

// ------------------------------------------------------------------ a2 keys --
// spread the low 10 bits of v so that bit b lands on bit 3b
__device__ __forceinline__ uint32_t ff_spread10(uint32_t v)
{
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

// Root cube from the bounding box, in the fp32 operation order of DESIGN.md (O3):
// S = max_a fl(hi_a - lo_a), S = 1 if 0; inv = fl(1024 / S).
__device__ __forceinline__ void ff_root_cube(const ff_globals* g, float lo[3], float& S, float& inv)
{
    S = 0.0f;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        lo[a] = ff_ord2f(g->bbox_ord[a]);
        float e = __fsub_rn(ff_ord2f(g->bbox_ord[4 + a]), lo[a]);
        S = fmaxf(S, e);
    }
    if (!(S > 0.0f)) S = 1.0f;
    inv = __fdiv_rn(1024.0f, S);
}

__global__ void __launch_bounds__(256) ff_k_keys(const float* __restrict__ pos, int n, ff_globals* g,
                                                 uint32_t* __restrict__ key)
{
    float lo[3], S, inv;
    ff_root_cube(g, lo, S, inv);
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) { g->lo[0] = lo[0]; g->lo[1] = lo[1]; g->lo[2] = lo[2]; g->S = S; g->inv = inv; }
    if (i >= n) return;
    uint32_t q[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float d = __fsub_rn(__ldg(pos + 3 * (size_t)i + a), lo[a]);
        int v = __float2int_rd(__fmul_rn(d, inv));      // floor, then to int
        q[a] = (uint32_t)min(1023, max(0, v));
    }
    key[i] = (ff_spread10(q[0]) << 2) | (ff_spread10(q[1]) << 1) | ff_spread10(q[2]);
}

// ------------------------------------------------------------ a3 radix sort --
// LSD, 8-bit digits, 4 passes over the 30-bit key.  Per pass: (1) per-tile digit
// histogram, (2) per-digit exclusive scan over tiles, (3) stable scatter using
// warp match ranking.  Stability within a tile: a warp owns a contiguous chunk
// and walks it in rounds of 32; rank = earlier rounds' count + lower lanes.
__global__ void __launch_bounds__(FF_SORT_THREADS)
ff_k_radix_hist(const uint32_t* __restrict__ key, int n, int shift, uint32_t mask,
                uint32_t* __restrict__ hist, int n_tiles)
{
    __shared__ uint32_t h[FF_RADIX];
    h[threadIdx.x] = 0;
    __syncthreads();
    int lane = ff_lane(), w = threadIdx.x >> 5;
    int base = blockIdx.x * FF_SORT_TILE + w * 32 * FF_SORT_ROUNDS;
#pragma unroll
    for (int r = 0; r < FF_SORT_ROUNDS; ++r) {
        int i = base + r * 32 + lane;
        bool valid = i < n;
        uint32_t d = valid ? ((__ldg(key + i) >> shift) & mask) : 0xffffffffu;
        unsigned peers = __match_any_sync(FF_FULL, d);
        if (valid && lane == __ffs(peers) - 1) atomicAdd(&h[d], (uint32_t)__popc(peers));
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * n_tiles + blockIdx.x] = h[threadIdx.x];
}

// one block per digit: exclusive scan of hist[d][0..n_tiles) in place, total -> g->digit_total[d]
__global__ void __launch_bounds__(256) ff_k_radix_scan(uint32_t* __restrict__ hist, int n_tiles, ff_globals* g)
{
    __shared__ uint32_t wsum[8];
    __shared__ uint32_t carry_s;
    uint32_t* row = hist + (size_t)blockIdx.x * n_tiles;
    int lane = ff_lane(), w = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < n_tiles; base += 256) {
        int i = base + threadIdx.x;
        uint32_t v = i < n_tiles ? row[i] : 0u;
        uint32_t x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(FF_FULL, x, o); if (lane >= o) x += y; }
        if (lane == 31) wsum[w] = x;
        __syncthreads();
        uint32_t woff = 0, tot = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) { uint32_t s = wsum[k]; if (k < w) woff += s; tot += s; }
        uint32_t carry = carry_s;
        if (i < n_tiles) row[i] = carry + woff + x - v;
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) g->digit_total[blockIdx.x] = carry_s;
}

__global__ void __launch_bounds__(FF_SORT_THREADS)
ff_k_radix_scatter(const uint32_t* __restrict__ kin, const uint32_t* __restrict__ vin,
                   uint32_t* __restrict__ kout, uint32_t* __restrict__ vout, int n, int shift, uint32_t mask,
                   const uint32_t* __restrict__ hist, int n_tiles, const ff_globals* __restrict__ g)
{
    __shared__ uint32_t wh[FF_SORT_THREADS / 32][FF_RADIX];   // per-warp digit counts, then bases
    __shared__ uint32_t wsum[8];
    int t = threadIdx.x, lane = t & 31, w = t >> 5;
#pragma unroll
    for (int k = 0; k < FF_SORT_THREADS / 32; ++k) wh[k][t] = 0;
    // exclusive scan of the digit totals -> first output slot of digit t
    uint32_t tot = g->digit_total[t], x = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(FF_FULL, x, o); if (lane >= o) x += y; }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    uint32_t dbase = x - tot;
#pragma unroll
    for (int k = 0; k < 8; ++k) if (k < w) dbase += wsum[k];

    uint32_t key[FF_SORT_ROUNDS], val[FF_SORT_ROUNDS], rank[FF_SORT_ROUNDS];
    int base = blockIdx.x * FF_SORT_TILE + w * 32 * FF_SORT_ROUNDS;
#pragma unroll
    for (int r = 0; r < FF_SORT_ROUNDS; ++r) {
        int i = base + r * 32 + lane;
        bool valid = i < n;
        key[r] = valid ? __ldg(kin + i) : 0xffffffffu;
        val[r] = valid ? (vin ? __ldg(vin + i) : (uint32_t)i) : 0u;
        uint32_t d = valid ? ((key[r] >> shift) & mask) : 0xffffffffu;
        unsigned peers = __match_any_sync(FF_FULL, d);
        int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if (valid && lane == leader) { old = wh[w][d]; wh[w][d] = old + (uint32_t)__popc(peers); }
        old = __shfl_sync(FF_FULL, old, leader);
        rank[r] = old + (uint32_t)__popc(peers & ((1u << lane) - 1u));
        __syncwarp();
    }
    __syncthreads();
    // digit t: global base of this tile, then exclusive prefix over the warps
    uint32_t run = dbase + hist[(size_t)t * n_tiles + blockIdx.x];
#pragma unroll
    for (int k = 0; k < FF_SORT_THREADS / 32; ++k) { uint32_t c = wh[k][t]; wh[k][t] = run; run += c; }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < FF_SORT_ROUNDS; ++r) {
        int i = base + r * 32 + lane;
        if (i < n) {
            uint32_t d = (key[r] >> shift) & mask;
            uint32_t dst = wh[w][d] + rank[r];
            kout[dst] = key[r];
            vout[dst] = val[r];
        }
    }
}

// sorted float4 copy of a caller-order [n][3] array: out[s] = in[perm[s]]
__global__ void __launch_bounds__(256) ff_k_gather4(const float* __restrict__ in, const uint32_t* __restrict__ perm,
                                                    int n, float4* __restrict__ out)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    size_t j = (size_t)__ldg(perm + s) * 3;
    out[s] = make_float4(__ldg(in + j), __ldg(in + j + 1), __ldg(in + j + 2), 0.0f);
}

int ff_launch_bbox_keys(ff_ctx* c, const float* pos)
{
    int n = (int)c->n;
    FF_LAUNCH(c, ff_k_reset, 1, 32, 0, c->g);
    int blocks = min((n + 255) / 256, c->num_sms * 8);
    FF_LAUNCH(c, ff_k_bbox, blocks, 256, 0, pos, n, c->g);
    FF_LAUNCH(c, ff_k_keys, (n + 255) / 256, 256, 0, pos, n, c->g, c->key[0]);
    return FF_OK;
}

int ff_launch_sort(ff_ctx* c, const float* pos)
{
    int n = (int)c->n;
    int n_tiles = (n + FF_SORT_TILE - 1) / FF_SORT_TILE;
    int cur = 0;
    for (int pass = 0; pass < 4; ++pass) {
        int shift = pass * FF_RADIX_BITS;
        uint32_t mask = pass == 3 ? 0x3fu : 0xffu;
        FF_LAUNCH(c, ff_k_radix_hist, n_tiles, FF_SORT_THREADS, 0, c->key[cur], n, shift, mask, c->sort_hist, n_tiles);
        FF_LAUNCH(c, ff_k_radix_scan, FF_RADIX, 256, 0, c->sort_hist, n_tiles, c->g);
        FF_LAUNCH(c, ff_k_radix_scatter, n_tiles, FF_SORT_THREADS, 0, c->key[cur],
                  pass == 0 ? (const uint32_t*)nullptr : c->idx[cur], c->key[cur ^ 1], c->idx[cur ^ 1], n, shift, mask,
                  c->sort_hist, n_tiles, c->g);
        cur ^= 1;
    }
    // four passes: the result is back in buffer 0
    FF_LAUNCH(c, ff_k_gather4, (n + 255) / 256, 256, 0, pos, c->idx[0], n, c->pos_s);
    return FF_OK;
}
