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
// Only after ff_create and after a call that failed half way: a completed build leaves this state behind itself
// (ff_k_build, phase 1).
__global__ void ff_k_reset(ff_globals* g)
{
    ff_reset_globals(g, threadIdx.x, blockDim.x);
    if (threadIdx.x == 0) g->n_cells = 0;
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

// Also: the digit histograms of all four sort passes (they do not depend on the order of the keys,
// so one read of the keys serves every pass) and the reset of the sort's tile-status words.
__global__ void __launch_bounds__(256) ff_k_keys(const float* __restrict__ pos, int n, ff_globals* g,
                                                 uint32_t* __restrict__ key, uint32_t* __restrict__ status,
                                                 int n_status)
{
    __shared__ uint32_t h[FF_SORT_PASSES][FF_RADIX];
#pragma unroll
    for (int p = 0; p < FF_SORT_PASSES; ++p) h[p][threadIdx.x] = 0;
    float lo[3], S, inv;
    ff_root_cube(g, lo, S, inv);
    const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
    if (tid == 0) { g->lo[0] = lo[0]; g->lo[1] = lo[1]; g->lo[2] = lo[2]; g->S = S; g->inv = inv; }
    for (int i = tid; i < n_status; i += nth) status[i] = 0u;
    __syncthreads();
    for (int i = tid; i < n; i += nth) {
        uint32_t q[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            float d = __fsub_rn(__ldg(pos + 3 * (size_t)i + a), lo[a]);
            int v = __float2int_rd(__fmul_rn(d, inv));      // floor, then to int
            FF_CHECK(g, v >= 0 && v <= 1024);
            q[a] = (uint32_t)min(1023, max(0, v));
        }
        const uint32_t k = (ff_spread10(q[0]) << 2) | (ff_spread10(q[1]) << 1) | ff_spread10(q[2]);
        key[i] = k;
#pragma unroll
        for (int p = 0; p < FF_SORT_PASSES; ++p) atomicAdd(&h[p][(k >> (p * FF_RADIX_BITS)) & (FF_RADIX - 1)], 1u);
    }
    __syncthreads();
#pragma unroll
    for (int p = 0; p < FF_SORT_PASSES; ++p)
        if (h[p][threadIdx.x]) atomicAdd(&g->digit_hist[p][threadIdx.x], h[p][threadIdx.x]);
}

// ------------------------------------------------------------ a3 radix sort --
// LSD, 8-bit digits, four passes over the 30-bit key, each pass ONE kernel that reads and writes
// every (key, index) pair once ("onesweep"): the global digit histograms come from ff_k_keys, and
// the offset of a tile inside a digit's output range is found by decoupled look-back over the
// status words of the earlier tiles (per tile and digit: count | state; a tile publishes its own
// count at once and its inclusive prefix as soon as it knows it).  Tiles are handed out by an
// atomic ticket, so every tile a block waits for is already running.  Stable: a warp owns a
// contiguous chunk and walks it in rounds of 32; rank = earlier tiles + earlier warps + earlier
// rounds + lower lanes with the same digit (peer mask from a shared-memory word per warp and digit).
#ifndef FF_SORT_WINDOW
#define FF_SORT_WINDOW 8
#endif
#define FF_ST_AGG 0x40000000u
#define FF_ST_PREFIX 0x80000000u
#define FF_ST_COUNT 0x3fffffffu

__global__ void __launch_bounds__(FF_SORT_THREADS)
ff_k_radix_onesweep(const uint32_t* __restrict__ kin, const uint32_t* __restrict__ vin,
                    uint32_t* __restrict__ kout, uint32_t* __restrict__ vout, int n, int pass,
                    uint32_t* status, ff_globals* g, const float* __restrict__ pos, float4* __restrict__ pos_s)
{
    __shared__ uint32_t wh[FF_SORT_THREADS / 32][FF_RADIX];   // per-warp digit counts, then offsets
    __shared__ uint32_t tile_base[FF_RADIX];
    __shared__ uint32_t skey[FF_SORT_TILE], sval[FF_SORT_TILE];
    __shared__ uint32_t wsum[8];
    __shared__ int s_tile;
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int shift = pass * FF_RADIX_BITS;
    if (t == 0) s_tile = atomicAdd(&g->sort_ticket[pass], 1);
#pragma unroll
    for (int k = 0; k < FF_SORT_THREADS / 32; ++k) wh[k][t] = 0;
    // exclusive scan of the global digit histogram -> first output slot of digit t
    uint32_t tot = g->digit_hist[pass][t], x = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(FF_FULL, x, o); if (lane >= o) x += y; }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    uint32_t dbase = x - tot;
#pragma unroll
    for (int k = 0; k < 8; ++k) if (k < w) dbase += wsum[k];
    const int tile = s_tile;
    FF_CHECK(g, tile >= 0 && tile * FF_SORT_TILE < n);

    uint32_t key[FF_SORT_ROUNDS], val[FF_SORT_ROUNDS], rank[FF_SORT_ROUNDS];
    const int base = tile * FF_SORT_TILE + w * 32 * FF_SORT_ROUNDS;
#pragma unroll
    for (int r = 0; r < FF_SORT_ROUNDS; ++r) {
        int i = base + r * 32 + lane;
        bool valid = i < n;
        key[r] = valid ? __ldg(kin + i) : 0xffffffffu;
        val[r] = valid ? (vin ? __ldg(vin + i) : (uint32_t)i) : 0u;
    }
    // Stable ranking inside the warp's chunk.  The lanes of a round that hold the same digit find each other through a
    // shared-memory word per (warp, digit): every lane ORs its lane bit in, reads the word back (= the peer mask), the
    // lowest peer bumps the warp's running count of that digit and clears the word for the next round.  One
    // shared-memory atomic per key instead of eight ballots with their mask arithmetic (the sort passes are
    // instruction bound, profiles/r2_hbm_phases.md).  The words live in `skey`, which is not needed before the
    // ranking is done.
    uint32_t* match = skey + w * FF_RADIX;
    static_assert(FF_SORT_TILE >= (FF_SORT_THREADS / 32) * FF_RADIX, "the match words of all warps fit in skey");
#pragma unroll
    for (int k = 0; k < FF_RADIX / 32; ++k) match[k * 32 + lane] = 0u;
    __syncwarp();
#pragma unroll
    for (int r = 0; r < FF_SORT_ROUNDS; ++r) {
        const bool valid = base + r * 32 + lane < n;
        const uint32_t d = (key[r] >> shift) & (FF_RADIX - 1);
        if (valid) atomicOr(&match[d], 1u << lane);
        __syncwarp();
        const unsigned peers = valid ? match[d] : 0u;
        const int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        __syncwarp();                                      // every peer has read the word before its leader clears it
        if (valid && lane == leader) { old = wh[w][d]; wh[w][d] = old + (uint32_t)__popc(peers); match[d] = 0u; }
        old = __shfl_sync(FF_FULL, old, leader < 0 ? 0 : leader);
        rank[r] = old + (uint32_t)__popc(peers & ((1u << lane) - 1u));
        __syncwarp();                                      // the cleared word before the next round's ORs
    }
    __syncthreads();
    // digit t: count of this tile; per-warp counts become offsets inside the tile's run of digit t
    uint32_t cnt = 0;
#pragma unroll
    for (int k = 0; k < FF_SORT_THREADS / 32; ++k) { uint32_t c = wh[k][t]; wh[k][t] = cnt; cnt += c; }
    // decoupled look-back: digits of this tile that precede ... = sum of the counts of tiles < tile
    volatile uint32_t* st = status + (size_t)tile * FF_RADIX + t;
    uint32_t excl = 0;
    if (tile == 0) {
        *st = cnt | FF_ST_PREFIX;
    } else {
        *st = cnt | FF_ST_AGG;
        // FF_SORT_WINDOW predecessors per step (independent loads: one memory latency per step, not per tile)
        int j = tile - 1;
        for (;;) {
            uint32_t v[FF_SORT_WINDOW];
#pragma unroll
            for (int q = 0; q < FF_SORT_WINDOW; ++q)
                v[q] = j - q >= 0 ? *(volatile uint32_t*)(status + (size_t)(j - q) * FF_RADIX + t) : FF_ST_PREFIX;
            bool done = false;
#pragma unroll
            for (int q = 0; q < FF_SORT_WINDOW; ++q) {
                if (done || !(v[q] & (FF_ST_PREFIX | FF_ST_AGG))) break;     // not published yet: re-read from here
                excl += v[q] & FF_ST_COUNT;
                --j;
                done = (v[q] & FF_ST_PREFIX) != 0;
            }
            if (done) break;
        }
        *st = (excl + cnt) | FF_ST_PREFIX;
    }
    // Reorder the tile by digit in shared memory, then write runs: consecutive threads write consecutive
    // slots of a digit's run (about 8 pairs = one 32-byte sector per run instead of one sector per pair).
    uint32_t lx = cnt;                                     // exclusive scan of the tile's digit counts
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(FF_FULL, lx, o); if (lane >= o) lx += y; }
    __syncthreads();                                       // wsum of the first scan fully read
    if (lane == 31) wsum[w] = lx;
    __syncthreads();
    uint32_t lstart = lx - cnt;
#pragma unroll
    for (int k = 0; k < 8; ++k) if (k < w) lstart += wsum[k];
    tile_base[t] = dbase + excl - lstart;                  // output slot of staged element i with digit t: tile_base[t] + i
#pragma unroll
    for (int k = 0; k < FF_SORT_THREADS / 32; ++k) wh[k][t] += lstart;   // staged position = wh[w][d] + rank
    __syncthreads();
#pragma unroll
    for (int r = 0; r < FF_SORT_ROUNDS; ++r) {
        if (base + r * 32 + lane < n) {
            uint32_t d = (key[r] >> shift) & (FF_RADIX - 1);
            uint32_t lp = wh[w][d] + rank[r];
            skey[lp] = key[r];
            sval[lp] = val[r];
        }
    }
    __syncthreads();
    const int tile_n = min(FF_SORT_TILE, n - tile * FF_SORT_TILE);
#pragma unroll
    for (int r = 0; r < FF_SORT_ROUNDS; ++r) {
        int i = r * FF_SORT_THREADS + t;
        if (i < tile_n) {
            uint32_t k = skey[i];
            uint32_t dst = tile_base[(k >> shift) & (FF_RADIX - 1)] + (uint32_t)i;
            const uint32_t v = sval[i];
            FF_CHECK(g, dst < (uint32_t)n && v < (uint32_t)n);
            kout[dst] = k;
            vout[dst] = v;
            // last pass: dst is the final sorted slot, so the sorted float4 positions are written here as well
            if (pos_s) pos_s[dst] = make_float4(__ldg(pos + 3 * (size_t)v), __ldg(pos + 3 * (size_t)v + 1), __ldg(pos + 3 * (size_t)v + 2), 0.0f);
        }
    }
}

int ff_launch_bbox_keys(ff_ctx* c, const float* pos)
{
    int n = (int)c->n;
    int n_tiles = (n + FF_SORT_TILE - 1) / FF_SORT_TILE;
    if (!c->globals_clean) FF_LAUNCH(c, ff_k_reset, 1, 256, 0, c->g);
    c->globals_clean = 0;                                  // until ff_k_build has been enqueued
    int blocks = min((n + 255) / 256, c->num_sms * 8);
    FF_LAUNCH(c, ff_k_bbox, blocks, 256, 0, pos, n, c->g);
    // every block ends with 1024 global atomics (its digit histograms): few blocks while the launch is latency
    // bound (measured: 2 per SM at 2^20, 8 per SM at 2^24)
    int kblocks = min((n + 255) / 256, c->num_sms * (n > (1 << 22) ? 8 : 2));
    FF_LAUNCH(c, ff_k_keys, kblocks, 256, 0, pos, n, c->g, c->key[0], c->sort_status, FF_SORT_PASSES * n_tiles * FF_RADIX);
    return FF_OK;
}

int ff_launch_sort(ff_ctx* c, const float* pos)
{
    int n = (int)c->n;
    int n_tiles = (n + FF_SORT_TILE - 1) / FF_SORT_TILE;
    int cur = 0;
    for (int pass = 0; pass < FF_SORT_PASSES; ++pass) {
        FF_LAUNCH(c, ff_k_radix_onesweep, n_tiles, FF_SORT_THREADS, 0, c->key[cur],
                  pass == 0 ? (const uint32_t*)nullptr : c->idx[cur], c->key[cur ^ 1], c->idx[cur ^ 1], n, pass,
                  c->sort_status + (size_t)pass * n_tiles * FF_RADIX, c->g,
                  pass == FF_SORT_PASSES - 1 ? pos : (const float*)nullptr,
                  pass == FF_SORT_PASSES - 1 ? c->pos_s : (float4*)nullptr);
        cur ^= 1;
    }
    // four passes: the result is back in buffer 0 (and the sorted positions are in pos_s)
    return FF_OK;
}
