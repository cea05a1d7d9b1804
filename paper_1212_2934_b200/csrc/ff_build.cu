// ff_build.cu -- a4 octree from the sorted Morton keys, a5 cell pseudo-particles.
//
// Paper: kernel 2 builds the octree by locked insertion and
// kernel 3 sums the cells bottom-up.  Here the tree of
// PAPER.md:147 ("divide into eight sub-cells while more than one particle") is
// read off the sorted 30-bit keys with no locks and no host round-trip:
//
//   L(i)  = octant digits shared by key[i-1] and key[i]        (L(0) := -1)
//   Lk(i) = digits shared by key[i] and key[i + N_leaf]        (-1 past the end)
//   the level-l cell that STARTS at slot i exists iff L(i) < l, and holds more
//   than N_leaf particles iff Lk(i) >= l; so the internal cells starting at i
//   are exactly the levels  L(i) < l <= min(Lk(i), 9).
//
// An exclusive scan of that count numbers the cells in pre-order, i.e. sorted by
// (first, level).  Children and ranges come from binary searches in the key array.
#include "ff_internal.cuh"
#include <cooperative_groups.h>
namespace cg = cooperative_groups;

#define FF_MOM_THREADS 256

__device__ __forceinline__ int ff_lprev(const uint32_t* __restrict__ key, int i)
{
    return i == 0 ? -1 : ff_common_levels(__ldg(key + i - 1), __ldg(key + i));
}

__device__ __forceinline__ int ff_cells_at(const uint32_t* __restrict__ key, int i, int n, int nleaf, int& lprev)
{
    lprev = ff_lprev(key, i);
    int lk = (i + nleaf < n) ? ff_common_levels(__ldg(key + i), __ldg(key + i + nleaf)) : -1;
    return max(0, min(lk, FF_MAX_LEVEL - 1) - lprev);
}

// ---- device-wide exclusive scan of ff_cells_at (reduce / scan block sums / write) --
__global__ void __launch_bounds__(FF_SCAN_THREADS)
ff_k_cells_reduce(const uint32_t* __restrict__ key, int n, int nleaf, uint32_t* __restrict__ blk)
{
    __shared__ uint32_t wsum[FF_SCAN_THREADS / 32];
    uint32_t s = 0;
    int base = blockIdx.x * FF_SCAN_TILE;
#pragma unroll
    for (int r = 0; r < FF_SCAN_ITEMS; ++r) {
        int i = base + r * FF_SCAN_THREADS + threadIdx.x;
        int lp;
        if (i < n) s += (uint32_t)ff_cells_at(key, i, n, nleaf, lp);
    }
    s = __reduce_add_sync(FF_FULL, s);
    if (ff_lane() == 0) wsum[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int k = 0; k < FF_SCAN_THREADS / 32; ++k) t += wsum[k];
        blk[blockIdx.x] = t;
    }
}

// single block: exclusive scan of blk[0..m) in place; total -> g->n_cells
__global__ void __launch_bounds__(1024) ff_k_scan_blocksums(uint32_t* __restrict__ blk, int m, ff_globals* g)
{
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t carry_s;
    int lane = ff_lane(), w = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < m; base += 1024) {
        int i = base + threadIdx.x;
        uint32_t v = i < m ? blk[i] : 0u, x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(FF_FULL, x, o); if (lane >= o) x += y; }
        if (lane == 31) wsum[w] = x;
        __syncthreads();
        uint32_t woff = 0, tot = 0;
        for (int k = 0; k < 32; ++k) { uint32_t s = wsum[k]; if (k < w) woff += s; tot += s; }
        uint32_t carry = carry_s;
        if (i < m) blk[i] = carry + woff + x - v;
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) g->n_cells = (int32_t)carry_s;
}

// per tile: exclusive scan in slot order (thread t owns FF_SCAN_ITEMS consecutive slots)
__global__ void __launch_bounds__(FF_SCAN_THREADS)
ff_k_cells_scan(const uint32_t* __restrict__ key, int n, int nleaf, const uint32_t* __restrict__ blk,
                int32_t* __restrict__ cell_base)
{
    __shared__ uint32_t wsum[FF_SCAN_THREADS / 32];
    int lane = ff_lane(), w = threadIdx.x >> 5;
    int first = blockIdx.x * FF_SCAN_TILE + threadIdx.x * FF_SCAN_ITEMS;
    uint32_t c[FF_SCAN_ITEMS], s = 0;
#pragma unroll
    for (int r = 0; r < FF_SCAN_ITEMS; ++r) {
        int i = first + r, lp;
        c[r] = i < n ? (uint32_t)ff_cells_at(key, i, n, nleaf, lp) : 0u;
        s += c[r];
    }
    uint32_t x = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(FF_FULL, x, o); if (lane >= o) x += y; }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    uint32_t run = blk[blockIdx.x] + x - s;
    for (int k = 0; k < w; ++k) run += wsum[k];
#pragma unroll
    for (int r = 0; r < FF_SCAN_ITEMS; ++r) {
        int i = first + r;
        if (i < n) cell_base[i] = (int32_t)run;
        run += c[r];
    }
}

// first slot in [lo, hi) whose key is >= bound (keys sorted ascending)
__device__ __forceinline__ int ff_lower_bound(const uint32_t* __restrict__ key, int lo, int hi, uint32_t bound)
{
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if (__ldg(key + mid) < bound) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// ---- a4: one thread per slot writes the internal cells that start there -----------
__global__ void __launch_bounds__(128)
ff_k_cells_fill(const uint32_t* __restrict__ key, int n, int nleaf, const int32_t* __restrict__ cell_base,
                int32_t* __restrict__ cell_first, int32_t* __restrict__ cell_end, int32_t* __restrict__ cell_level,
                int32_t* __restrict__ cell_child, int32_t* __restrict__ leaf_count, int cell_cap, ff_globals* g)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int lprev;
    int cnt = ff_cells_at(key, i, n, nleaf, lprev);
    {   // deepest level holding an internal cell (bounds the level loop of ff_k_moments)
        int deepest = __reduce_max_sync(__activemask(), cnt > 0 ? lprev + cnt : 0);
        if (ff_lane() == 0 && deepest > 0) atomicMax(&g->max_level, deepest);
    }
    if (cnt == 0) return;
    int base = cell_base[i];
    if (base + cnt > cell_cap) { g->error = FF_ERR_CAPACITY; return; }
    uint32_t k = __ldg(key + i);
    int end_parent = n;                                    // end of the enclosing cell: search bound
    for (int q = 0; q < cnt; ++q) {
        int l = lprev + 1 + q;
        int id = base + q;
        int sh = 3 * (FF_MAX_LEVEL - l);                   // bits below the level-l prefix
        int end;
        if (l == 0) end = n;
        else {
            uint32_t bound = ((k >> sh) + 1u) << sh;       // first key past this cell (no overflow: 30-bit keys)
            end = ff_lower_bound(key, i + 1, end_parent, bound);
        }
        end_parent = end;
        cell_first[id] = i;
        cell_end[id] = end;
        cell_level[id] = l;
        // children: octant boundaries inside [i, end)
        int csh = sh - 3;
        uint32_t cpre = (k >> sh) << 3;                    // child prefix without the octant
        int b = i;
        for (int o = 0; o < 8; ++o) {
            int e = (o == 7) ? end : ff_lower_bound(key, b, end, (cpre + (uint32_t)o + 1u) << csh);
            int cc = e - b;
            int32_t ent;
            if (cc == 0) ent = FF_CHILD_EMPTY;
            else if (cc > nleaf && l + 1 < FF_MAX_LEVEL) {
                // internal child: starts at slot b on level l+1
                int lp = ff_lprev(key, b);
                ent = cell_base[b] + (l + 1 - lp - 1);
            } else if (cc == 1) ent = (int32_t)(FF_CHILD_LEAF1 | (uint32_t)b);
            else { ent = (int32_t)(FF_CHILD_LEAF1 | FF_CHILD_MULTI | (uint32_t)b); leaf_count[b] = cc; }
            cell_child[8 * (size_t)id + o] = ent;
            b = e;
        }
    }
}

// ---- a5: Eq. 14: ONE cooperative launch -----------------------
// Phase 0 gathers the moments into sorted float4 order; then the levels are summed deepest
// first with a grid-wide barrier between levels (the paper's kernel 3 lets threads spin on
// their children instead; ten launches cost ~14 us each at N = 2^20).
// fp64 sums in the fixed order of DESIGN.md (O4): children in octant order,
// ((c0 + c1) + c2) + ...; a leaf's particles left to right; one fp64 divide and a
// single rounding to fp32.
__global__ void __launch_bounds__(FF_MOM_THREADS)
ff_k_moments(const float* __restrict__ mom, const uint32_t* __restrict__ perm, int n, ff_globals* __restrict__ g,
             const int32_t* __restrict__ cell_first, const int32_t* __restrict__ cell_end,
             const int32_t* __restrict__ cell_level, const int32_t* __restrict__ cell_child,
             const int32_t* __restrict__ leaf_count, const float4* __restrict__ pos_s, float4* __restrict__ mom_s,
             double* __restrict__ sum_u, double* __restrict__ sum_p, float4* __restrict__ centre,
             float4* __restrict__ moment)
{
    cg::grid_group grid = cg::this_grid();
    const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
    for (int s = tid; s < n; s += nth) {
        size_t j = (size_t)__ldg(perm + s) * 3;
        mom_s[s] = make_float4(__ldg(mom + j), __ldg(mom + j + 1), __ldg(mom + j + 2), 0.0f);
    }
    if (tid == 0) g->walk_next = 0;                        // the walk's group counter (this is the last launch before it)
    const int n_cells = g->n_cells;
    const int top = min(g->max_level, FF_MAX_LEVEL - 1);   // deepest level that holds an internal cell
    const float S = g->S;
    // Eight lanes per cell: lane o loads child o (one exposed memory latency per cell instead of eight),
    // parks its six fp64 sums in shared memory, then lane a < 6 adds component a over the children in
    // octant order -- the same ((c0 + c1) + c2) + ... as a sequential loop.
    __shared__ double sh[FF_MOM_THREADS / 8][8][6];
    const int o = threadIdx.x & 7;
    const unsigned gshift = (threadIdx.x & 24);            // first lane of this group inside the warp
    const unsigned gmask = 0xffu << gshift;
    double(*mine)[6] = sh[threadIdx.x >> 3];
    const int gid = tid >> 3, ngroups = nth >> 3;
    grid.sync();
    for (int level = top; level >= 0; --level) {
        const float s = ldexpf(S, -level);
        const float s2 = __fmul_rn(s, s);
        for (int id = gid; id < n_cells; id += ngroups) {
            if (cell_level[id] != level) continue;         // uniform over the group's eight lanes
            const int32_t e = cell_child[8 * (size_t)id + o];
            const bool have = e != FF_CHILD_EMPTY;
            if (e >= 0) {
                // plain loads: written earlier in this launch by other blocks (ordered by grid.sync)
#pragma unroll
                for (int a = 0; a < 3; ++a) { mine[o][a] = sum_u[3 * (size_t)e + a]; mine[o][3 + a] = sum_p[3 * (size_t)e + a]; }
            } else if (have) {
                int slot = (int)((uint32_t)e & FF_CHILD_SLOT);
                int cc = ((uint32_t)e & FF_CHILD_MULTI) ? leaf_count[slot] : 1;
                float4 p = pos_s[slot], m = mom_s[slot];
                double cu[3] = { m.x, m.y, m.z }, cp[3] = { p.x, p.y, p.z };
                for (int j = slot + 1; j < slot + cc; ++j) {
                    p = pos_s[j]; m = mom_s[j];
                    cu[0] += (double)m.x; cu[1] += (double)m.y; cu[2] += (double)m.z;
                    cp[0] += (double)p.x; cp[1] += (double)p.y; cp[2] += (double)p.z;
                }
#pragma unroll
                for (int a = 0; a < 3; ++a) { mine[o][a] = cu[a]; mine[o][3 + a] = cp[a]; }
            }
            const unsigned present = (__ballot_sync(gmask, have) >> gshift) & 0xffu;   // also orders the smem writes
            const double cnt = (double)(cell_end[id] - cell_first[id]);
            double t = 0.0;
            if (o < 6) {
                bool started = false;
#pragma unroll
                for (int c = 0; c < 8; ++c)
                    if (present & (1u << c)) { t = started ? t + mine[c][o] : mine[c][o]; started = true; }
                if (o < 3) sum_u[3 * (size_t)id + o] = t; else sum_p[3 * (size_t)id + (o - 3)] = t;
            }
            float* cen = reinterpret_cast<float*>(centre + id);
            float* mo = reinterpret_cast<float*>(moment + id);
            if (o < 3) mo[o] = (float)t;
            else if (o < 6) cen[o - 3] = (float)(t / cnt);
            else if (o == 6) cen[3] = s2;
            else mo[3] = (float)cnt;
            __syncwarp(gmask);                             // smem slots are reused by the group's next cell
        }
        if (level > 0) grid.sync();
    }
}

int ff_launch_build(ff_ctx* c)
{
    int n = (int)c->n;
    int tiles = (n + FF_SCAN_TILE - 1) / FF_SCAN_TILE;
    FF_LAUNCH(c, ff_k_cells_reduce, tiles, FF_SCAN_THREADS, 0, c->key[0], n, c->nleaf, c->scan_blk);
    FF_LAUNCH(c, ff_k_scan_blocksums, 1, 1024, 0, c->scan_blk, tiles, c->g);
    FF_LAUNCH(c, ff_k_cells_scan, tiles, FF_SCAN_THREADS, 0, c->key[0], n, c->nleaf, c->scan_blk, c->cell_base);
    FF_LAUNCH(c, ff_k_cells_fill, (n + 127) / 128, 128, 0, c->key[0], n, c->nleaf, c->cell_base, c->cell_first,
              c->cell_end, c->cell_level, c->cell_child, c->leaf_count, (int)c->cell_cap, c->g);
    return FF_OK;
}

int ff_launch_moments(ff_ctx* c, const float* mom)
{
    int n = (int)c->n;
    static int per_sm = 0;
    if (!per_sm) {
        FF_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ff_k_moments, FF_MOM_THREADS, 0));
        if (per_sm < 1) return FF_ERR_CUDA;
    }
    int blocks = min((n + FF_MOM_THREADS - 1) / FF_MOM_THREADS, c->num_sms * min(per_sm, 8));
    const uint32_t* perm = c->idx[0];
    void* args[] = { (void*)&mom, (void*)&perm, (void*)&n, (void*)&c->g, (void*)&c->cell_first, (void*)&c->cell_end,
                     (void*)&c->cell_level, (void*)&c->cell_child, (void*)&c->leaf_count, (void*)&c->pos_s,
                     (void*)&c->mom_s, (void*)&c->cell_sum_u, (void*)&c->cell_sum_p, (void*)&c->cell_centre,
                     (void*)&c->cell_moment };
    FF_CUDA(c, cudaLaunchCooperativeKernel((const void*)ff_k_moments, dim3(blocks), dim3(FF_MOM_THREADS), args, 0,
                                           c->stream));
    c->launches++;
    return FF_OK;
}
