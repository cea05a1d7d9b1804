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

#ifndef FF_MOM_THREADS
#define FF_MOM_THREADS 512
#endif
#define FF_MOM_SOLO 1                 // levels 0..1 of the moment pass run in one block
#ifndef FF_BUILD_THREADS
#define FF_BUILD_THREADS 512
#endif
#define FF_BUILD_ITEMS 8
#define FF_BUILD_TILE (FF_BUILD_THREADS * FF_BUILD_ITEMS)

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

// first slot in [lo, hi) whose key is >= bound (keys sorted ascending)
__device__ __forceinline__ int ff_lower_bound(const uint32_t* __restrict__ key, int lo, int hi, uint32_t bound)
{
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if (__ldg(key + mid) < bound) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// the same, galloping up from lo: ~2 log2(answer - lo) probes, short for the many small cells
__device__ __forceinline__ int ff_gallop_bound(const uint32_t* __restrict__ key, int lo, int n, uint32_t bound)
{
    int pos = lo, step = 1;
    while (pos < n && __ldg(key + pos) < bound) { lo = pos + 1; pos += step; step <<= 1; }
    return ff_lower_bound(key, lo, min(pos, n), bound);
}

// ---- a4: the whole octree build as ONE cooperative launch ---------------------------------
//   phase 1  every block counts the cells that start in its contiguous range of slots
//   phase 2  exclusive scan (block prefix + in-tile scan) -> cell_base[slot]; every cell gets
//            its first slot and level; level histogram
//   phase 3  eight lanes per cell (lane o = octant o).  The group reads a WINDOW of the 32 sorted
//            keys that follow the cell's first slot in one coalesced step and counts, per octant
//            bound, the window keys below it (byte counters packed in two words, summed over the
//            eight lanes with three shuffles): for the ~95 % of the cells that hold <= 32
//            particles this gives every child boundary after ONE memory latency.  An octant whose
//            end lies beyond the window falls back to a galloping search from the window's end.
//            Then range and child links (non-empty sub-cells compacted to the front, in octant
//            order); the cell's id is appended to its level's list (ff_k_moments walks the levels
//            deepest first).
// The paper builds the tree by locked insertion (kernel 2); no locks here, and
// the result does not depend on scheduling except for the order inside a level list, which no
// result depends on.
#define FF_BUILD_WINDOW 32
#ifndef FF_BUILD_CELLS
#define FF_BUILD_CELLS 4                  // cells a group of eight lanes has in flight (phase 3)
#endif
__global__ void __launch_bounds__(FF_BUILD_THREADS)
ff_k_build(const uint32_t* __restrict__ key, int n, int nleaf, uint32_t* __restrict__ blk,
           int32_t* __restrict__ cell_base, int32_t* __restrict__ cell_first, int32_t* __restrict__ cell_end,
           int32_t* __restrict__ cell_level, int32_t* __restrict__ cell_child, int4* __restrict__ cell_info,
           int32_t* __restrict__ leaf_count, int32_t* __restrict__ cell_list, int cell_cap, ff_globals* g)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ uint32_t wsum[FF_BUILD_THREADS / 32];
    __shared__ uint32_t s_bcast[2];
    __shared__ int s_hist[FF_MAX_LEVEL], s_cur[FF_MAX_LEVEL];
    const int lane = ff_lane(), w = threadIdx.x >> 5;
    const int tiles = (n + FF_BUILD_TILE - 1) / FF_BUILD_TILE;
    const int tpb = (tiles + gridDim.x - 1) / gridDim.x;
    const int t0 = min(tiles, (int)blockIdx.x * tpb), t1 = min(tiles, t0 + tpb);

    // ---- phase 1
    {
        uint32_t s = 0;
        for (int t = t0; t < t1; ++t) {
#pragma unroll
            for (int r = 0; r < FF_BUILD_ITEMS; ++r) {
                int i = t * FF_BUILD_TILE + r * FF_BUILD_THREADS + threadIdx.x, lp;
                if (i < n) s += (uint32_t)ff_cells_at(key, i, n, nleaf, lp);
            }
        }
        s = __reduce_add_sync(FF_FULL, s);
        if (lane == 0) wsum[w] = s;
        __syncthreads();
        if (threadIdx.x == 0) {
            uint32_t t = 0;
            for (int k = 0; k < FF_BUILD_THREADS / 32; ++k) t += wsum[k];
            blk[blockIdx.x] = t;
        }
    }
    // the state the NEXT ff_build_tree starts from (bounding box, sort tickets and digit histograms are all consumed
    // by now): saves a reset launch per step; ff_create and a failed call run ff_k_reset instead
    if (blockIdx.x == gridDim.x - 1) ff_reset_globals(g, threadIdx.x, FF_BUILD_THREADS);
    grid.sync();

    // ---- phase 2
    {
        uint32_t before = 0, total = 0;
        for (int j = threadIdx.x; j < (int)gridDim.x; j += FF_BUILD_THREADS) {
            uint32_t v = blk[j];
            total += v;
            if (j < (int)blockIdx.x) before += v;
        }
        before = __reduce_add_sync(FF_FULL, before);
        total = __reduce_add_sync(FF_FULL, total);
        __syncthreads();
        if (threadIdx.x < 2) s_bcast[threadIdx.x] = 0;
        if (threadIdx.x < FF_MAX_LEVEL) s_hist[threadIdx.x] = 0;
        __syncthreads();
        if (lane == 0) { atomicAdd(&s_bcast[0], before); atomicAdd(&s_bcast[1], total); }
        __syncthreads();
        uint32_t carry = s_bcast[0];
        total = s_bcast[1];
        const bool fits = total <= (uint32_t)cell_cap;
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            g->n_cells = fits ? (int32_t)total : 0;
            if (!fits) g->error = FF_ERR_CAPACITY;
        }
        for (int t = t0; t < t1; ++t) {
            const int first = t * FF_BUILD_TILE + threadIdx.x * FF_BUILD_ITEMS;
            uint32_t c[FF_BUILD_ITEMS], s = 0;
            int lp[FF_BUILD_ITEMS];
#pragma unroll
            for (int r = 0; r < FF_BUILD_ITEMS; ++r) {
                int i = first + r;
                lp[r] = 0;
                c[r] = i < n ? (uint32_t)ff_cells_at(key, i, n, nleaf, lp[r]) : 0u;
                s += c[r];
            }
            uint32_t x = s;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(FF_FULL, x, o); if (lane >= o) x += y; }
            __syncthreads();                               // wsum of the previous tile fully read
            if (lane == 31) wsum[w] = x;
            __syncthreads();
            uint32_t run = carry + x - s, tile_total = 0;
            for (int k = 0; k < FF_BUILD_THREADS / 32; ++k) { uint32_t v = wsum[k]; if (k < w) run += v; tile_total += v; }
#pragma unroll
            for (int r = 0; r < FF_BUILD_ITEMS; ++r) {
                int i = first + r;
                if (i < n) cell_base[i] = (int32_t)run;
                if (fits)
                    for (uint32_t q = 0; q < c[r]; ++q) {
                        const int l = lp[r] + 1 + (int)q;
                        FF_CHECK(g, run + q < (uint32_t)cell_cap && l >= 0 && l < FF_MAX_LEVEL);
                        cell_first[run + q] = i;
                        cell_level[run + q] = l;
                        atomicAdd(&s_hist[l], 1);
                    }
                run += c[r];
            }
            carry += tile_total;
        }
        __syncthreads();
        if (threadIdx.x < FF_MAX_LEVEL && s_hist[threadIdx.x]) atomicAdd(&g->level_count[threadIdx.x], s_hist[threadIdx.x]);
    }
    grid.sync();

    // ---- phase 3
    // Latency bound (three dependent loads per cell: first slot -> window keys -> cell_base of the children), so every
    // group of eight lanes works on FF_BUILD_CELLS cells at a time and issues each stage's loads for all of them together.
    const int n_cells = g->n_cells;
    const int o = threadIdx.x & 7;
    const int gsh = threadIdx.x & 24;
    const unsigned gmask = 0xffu << gsh;
    const int stride = gridDim.x * (FF_BUILD_THREADS / 8);
    const int id0 = blockIdx.x * (FF_BUILD_THREADS / 8) + (threadIdx.x >> 3);
    // cell ids grouped by level (ff_k_moments walks the levels deepest first): start of every level's list, then
    // the block reserves, per level, room for the cells it is about to handle (one global atomic per level and block)
    __syncthreads();
    if (threadIdx.x == 0) {
        int run = 0, deepest = 0;
        for (int l = 0; l < FF_MAX_LEVEL; ++l) {
            s_cur[l] = run;                                // start of level l in cell_list
            if (blockIdx.x == 0) g->level_start[l] = run;
            int cnt = g->level_count[l];
            if (cnt > 0) deepest = l;
            run += cnt;
        }
        if (blockIdx.x == 0) { g->level_start[FF_MAX_LEVEL] = run; g->max_level = deepest; }
    }
    if (threadIdx.x < FF_MAX_LEVEL) s_hist[threadIdx.x] = 0;
    __syncthreads();
    for (int id = id0; id < n_cells; id += stride)
        if (o == 0) atomicAdd(&s_hist[cell_level[id]], 1);
    __syncthreads();
    if (threadIdx.x < FF_MAX_LEVEL && s_hist[threadIdx.x])
        s_cur[threadIdx.x] += atomicAdd(&g->level_cursor[threadIdx.x], s_hist[threadIdx.x]);
    __syncthreads();
    constexpr int U = FF_BUILD_CELLS, R = FF_BUILD_WINDOW / 8;
    for (int base_id = id0; base_id < n_cells; base_id += U * stride) {
        int first[U], l[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int id = base_id + u * stride;
            first[u] = id < n_cells ? cell_first[id] : 0;
            l[u] = id < n_cells ? cell_level[id] : 0;
        }
        // the windows: lane o holds the keys of slots first + o + 8 r; slots past the end count as "beyond the cell"
        uint32_t kw[U][R];
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int i = first[u] + o + 8 * r;
                kw[u][r] = (base_id + u * stride < n_cells && i < n) ? __ldg(key + i) : 0xffffffffu;
            }
        int e[U], b[U];
        int32_t ent[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int sh = 3 * (FF_MAX_LEVEL - l[u]);      // bits below the level-l prefix
            const int csh = sh - 3;
            const uint32_t k = __shfl_sync(gmask, kw[u][0], 0, 8);
            const uint32_t pre = k >> sh;
            // byte o' of (lo, hi) = number of this lane's window keys whose octant inside the cell is <= o'
            uint32_t lo = 0, hi = 0;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const bool inside = (kw[u][r] >> sh) == pre;
                const uint32_t c = (kw[u][r] >> csh) & 7u;
                if (inside) {
                    if (c < 4u) { lo += 0x01010101u << (8u * c); hi += 0x01010101u; }
                    else hi += 0x01010101u << (8u * (c - 4u));
                }
            }
#pragma unroll
            for (int d = 1; d < 8; d <<= 1) {
                lo += __shfl_xor_sync(gmask, lo, d, 8);
                hi += __shfl_xor_sync(gmask, hi, d, 8);
            }
            const int below = (int)(((o < 4 ? lo : hi) >> (8 * (o & 3))) & 0xffu);   // window keys in octants <= o
            e[u] = first[u] + below;
            // every window key lies in octants <= o: the end of octant o is beyond the window
            // (no overflow in the bound: 30-bit keys, the largest bound is 1 << 30)
            if (below == FF_BUILD_WINDOW)
                e[u] = ff_gallop_bound(key, first[u] + FF_BUILD_WINDOW, n, ((pre << 3) + (uint32_t)o + 1u) << csh);
            b[u] = __shfl_up_sync(gmask, e[u], 1, 8);
            if (o == 0) b[u] = first[u];
            // an internal child = the level l+1 cell that starts at slot b.  Cells that start at the same slot are
            // numbered consecutively by level, so a child starting at this cell's own first slot is id + 1; any other
            // child is the first cell starting at its slot (L(b) = l there): cell_base[b]
            const bool internal = e[u] - b[u] > nleaf && l[u] + 1 < FF_MAX_LEVEL;
            ent[u] = (internal && b[u] != first[u]) ? cell_base[b[u]] : base_id + u * stride + 1;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int id = base_id + u * stride;
            if (id >= n_cells) break;
            const int cc = e[u] - b[u];
            const bool internal = cc > nleaf && l[u] + 1 < FF_MAX_LEVEL;
            int32_t en = ent[u];
            FF_CHECK(g, first[u] <= b[u] && b[u] <= e[u] && e[u] <= n && (o != 7 || e[u] > first[u]));
            FF_CHECK(g, !(cc != 0 && internal) || (en > id && en < n_cells));
            if (cc == 0) en = FF_CHILD_EMPTY;
            else if (internal) ;
            else if (cc == 1) en = (int32_t)(FF_CHILD_LEAF1 | (uint32_t)b[u]);
            else { en = (int32_t)(FF_CHILD_LEAF1 | FF_CHILD_MULTI | (uint32_t)b[u]); leaf_count[b[u]] = cc; }
            // the eight links are stored COMPACTED: the non-empty sub-cells first, in octant order, then the empty ones
            // (the walk pushes the first n_children links without looking at them; the moments add them in this order)
            const unsigned present = (__ballot_sync(gmask, cc != 0) >> gsh) & 0xffu;
            const int nch = __popc(present);
            const int rank = __popc(present & ((1u << o) - 1u));
            cell_child[8 * (size_t)id + (cc != 0 ? rank : nch + (o - rank))] = en;
            if (o == 7) { cell_end[id] = e[u]; cell_info[id] = make_int4(first[u], e[u], nch, l[u]); }
            if (o == 0) {
                const int at = atomicAdd(&s_cur[l[u]], 1);
                FF_CHECK(g, at >= 0 && at < n_cells);
                cell_list[at] = id;
            }
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
// QUAD (FF_OPT_CELL_ORDER = 1): also the cell tensor D = sum_i (rho_i - rho') (x) u_i, symmetric part,
// from six more fp64 sums of the symmetrised products rho_i (x) u_i in the same fixed order (O4b); every fp64
// operation is an explicit round-to-nearest intrinsic so that no FMA contraction changes a bit against the oracle.
__device__ __forceinline__ void ff_sym_products(const float4& p, const float4& m, double out[6])
{
    const double px = p.x, py = p.y, pz = p.z, ux = m.x, uy = m.y, uz = m.z;
    out[0] = __dmul_rn(px, ux); out[1] = __dmul_rn(py, uy); out[2] = __dmul_rn(pz, uz);
    out[3] = __dmul_rn(__dadd_rn(__dmul_rn(px, uy), __dmul_rn(py, ux)), 0.5);
    out[4] = __dmul_rn(__dadd_rn(__dmul_rn(px, uz), __dmul_rn(pz, ux)), 0.5);
    out[5] = __dmul_rn(__dadd_rn(__dmul_rn(py, uz), __dmul_rn(pz, uy)), 0.5);
}

template <bool QUAD>
__global__ void __launch_bounds__(FF_MOM_THREADS)
ff_k_moments(const float* __restrict__ mom, const uint32_t* __restrict__ perm, int n, ff_globals* __restrict__ g,
             const int32_t* __restrict__ cell_first, const int32_t* __restrict__ cell_end,
             const int32_t* __restrict__ cell_list, const int32_t* __restrict__ cell_child,
             const int32_t* __restrict__ leaf_count, const float4* __restrict__ pos_s, float4* __restrict__ mom_s,
             double* __restrict__ sums, float4* __restrict__ centre,
             float4* __restrict__ moment, double* __restrict__ sums2, float4* __restrict__ quad)
{
    constexpr int NS = QUAD ? 12 : 6;                      // fp64 sums per cell
    cg::grid_group grid = cg::this_grid();
    const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
    for (int s = tid; s < n; s += nth) {
        size_t j = (size_t)__ldg(perm + s) * 3;
        mom_s[s] = make_float4(__ldg(mom + j), __ldg(mom + j + 1), __ldg(mom + j + 2), 0.0f);
    }
    if (tid == 0) g->walk_next = 0;                        // the walk's group counter (this is the last launch before it)
    const int top = min(g->max_level, FF_MAX_LEVEL - 1);   // deepest level that holds an internal cell
    const float S = g->S;
    // Eight lanes per cell: lane o loads child o (one exposed memory latency per cell instead of eight),
    // parks its fp64 sums in shared memory, then lane a < 6 adds component a (and a + 6) over the children in
    // octant order -- the same ((c0 + c1) + c2) + ... as a sequential loop.
    __shared__ double sh[FF_MOM_THREADS / 8][8][NS];
    const int o = threadIdx.x & 7;
    const unsigned gshift = (threadIdx.x & 24);            // first lane of this group inside the warp
    const unsigned gmask = 0xffu << gshift;
    double(*mine)[NS] = sh[threadIdx.x >> 3];
    const int gid = tid >> 3, ngroups = nth >> 3;
    grid.sync();
    for (int level = top; level >= 0; --level) {
        // the nine cells of levels 0..FF_MOM_SOLO are left to block 0 alone: block-wide barriers
        // instead of two more grid-wide ones (more levels than that cost more in one block than the barriers)
        const bool solo = level <= FF_MOM_SOLO;
        if (solo && blockIdx.x != 0) break;
        const float s = ldexpf(S, -level);
        const float s2 = __fmul_rn(s, s);
        const int ls = g->level_start[level], le = g->level_start[level + 1];
        const int kstep = solo ? FF_MOM_THREADS / 8 : ngroups;
        // software pipeline over the dependent loads list -> child link -> child data: the cell id is fetched two
        // iterations ahead and the child link one ahead, so that an iteration exposes one memory latency, not three
        const int k0 = ls + (solo ? (int)(threadIdx.x >> 3) : gid);
        int id1 = k0 < le ? cell_list[k0] : -1;                        // cell of the coming iteration
        int id2 = k0 + kstep < le ? cell_list[k0 + kstep] : -1;        // and of the one after
        int32_t e1 = id1 >= 0 ? cell_child[8 * (size_t)id1 + o] : FF_CHILD_EMPTY;
        for (int k = k0; k < le; k += kstep) {
            const int id = id1;
            const int32_t e = e1;
            FF_CHECK(g, id >= 0 && id < g->n_cells && (e < 0 || (e > id && e < g->n_cells)));
            id1 = id2;
            id2 = k + 2 * kstep < le ? cell_list[k + 2 * kstep] : -1;
            e1 = id1 >= 0 ? cell_child[8 * (size_t)id1 + o] : FF_CHILD_EMPTY;
            const bool have = e != FF_CHILD_EMPTY;
            if (e >= 0) {
                // plain loads: written earlier in this launch by other blocks (ordered by grid.sync)
#pragma unroll
                for (int a = 0; a < 6; a += 2) {           // one 64-byte record per cell: u.xyz, p.xyz (two sectors)
                    const double2 v = *reinterpret_cast<const double2*>(sums + 8 * (size_t)e + a);
                    mine[o][a] = v.x; mine[o][a + 1] = v.y;
                    if (QUAD) {
                        const double2 q = *reinterpret_cast<const double2*>(sums2 + 8 * (size_t)e + a);
                        mine[o][6 + a] = q.x; mine[o][7 + a] = q.y;
                    }
                }
            } else if (have) {
                int slot = (int)((uint32_t)e & FF_CHILD_SLOT);
                int cc = ((uint32_t)e & FF_CHILD_MULTI) ? leaf_count[slot] : 1;
                float4 p = pos_s[slot], m = mom_s[slot];
                double cu[3] = { m.x, m.y, m.z }, cp[3] = { p.x, p.y, p.z }, cq[6];
                if (QUAD) ff_sym_products(p, m, cq);
                for (int j = slot + 1; j < slot + cc; ++j) {
                    p = pos_s[j]; m = mom_s[j];
                    cu[0] += (double)m.x; cu[1] += (double)m.y; cu[2] += (double)m.z;
                    cp[0] += (double)p.x; cp[1] += (double)p.y; cp[2] += (double)p.z;
                    if (QUAD) {
                        double pq[6];
                        ff_sym_products(p, m, pq);
#pragma unroll
                        for (int a = 0; a < 6; ++a) cq[a] = __dadd_rn(cq[a], pq[a]);
                    }
                }
#pragma unroll
                for (int a = 0; a < 3; ++a) { mine[o][a] = cu[a]; mine[o][3 + a] = cp[a]; }
                if (QUAD) {
#pragma unroll
                    for (int a = 0; a < 6; ++a) mine[o][6 + a] = cq[a];
                }
            }
            const unsigned present = (__ballot_sync(gmask, have) >> gshift) & 0xffu;   // also orders the smem writes
            const double cnt = (double)(cell_end[id] - cell_first[id]);
            double t = 0.0, t2 = 0.0;
            if (o < 6) {
                bool started = false;
#pragma unroll
                for (int c = 0; c < 8; ++c)
                    if (present & (1u << c)) {
                        t = started ? t + mine[c][o] : mine[c][o];
                        if (QUAD) t2 = started ? __dadd_rn(t2, mine[c][6 + o]) : mine[c][6 + o];
                        started = true;
                    }
                sums[8 * (size_t)id + o] = t;
                if (QUAD) sums2[8 * (size_t)id + o] = t2;
            }
            float* cen = reinterpret_cast<float*>(centre + id);
            float* mo = reinterpret_cast<float*>(moment + id);
            if (o < 3) mo[o] = (float)t;
            else if (o < 6) cen[o - 3] = (float)(t / cnt);
            else if (o == 6) cen[3] = s2;
            else mo[3] = (float)cnt;
            if (QUAD) {
                // lane c < 6 holds component c of D in the order xx yy zz xy xz yz = (ia, ib); su_a sits in lane a, sp_a
                // in lane 3 + a of this group of eight
                const int ia = o < 3 ? o : (o == 5 ? 1 : 0), ib = o < 3 ? o : (o == 3 ? 1 : 2);
                const double su_a = __shfl_sync(gmask, t, ia, 8), su_b = __shfl_sync(gmask, t, ib, 8);
                const double cen_a = __ddiv_rn(__shfl_sync(gmask, t, 3 + ia, 8), cnt);
                const double cen_b = __ddiv_rn(__shfl_sync(gmask, t, 3 + ib, 8), cnt);
                const double cu = o < 3 ? __dmul_rn(cen_a, su_b)
                                        : __dmul_rn(__dadd_rn(__dmul_rn(cen_a, su_b), __dmul_rn(cen_b, su_a)), 0.5);
                reinterpret_cast<float*>(quad + 2 * (size_t)id)[o] = o < 6 ? (float)__dsub_rn(t2, cu) : 0.0f;
            }
            __syncwarp(gmask);                             // smem slots are reused by the group's next cell
        }
        if (level > FF_MOM_SOLO) grid.sync();
        else if (level > 0) __syncthreads();
    }
}

int ff_launch_build(ff_ctx* c)
{
    int n = (int)c->n;
    int& per_sm = c->occ_build;                            // per context: contexts may live on different devices
    if (!per_sm) {
        FF_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ff_k_build, FF_BUILD_THREADS, 0));
        if (per_sm < 1) return FF_ERR_CUDA;
    }
    // phase 3 is latency bound and wants every thread slot of the GPU; a small n gets as many blocks as it has
    // groups of 32 particles (a block with no tile skips phases 1-2)
    int blocks = max(1, min(min((n + 31) / 32, c->num_sms * min(per_sm, 8)), FF_BUILD_MAX_BLOCKS));
    int nleaf = c->nleaf, cap = (int)c->cell_cap;
    void* args[] = { (void*)&c->key[0], (void*)&n, (void*)&nleaf, (void*)&c->scan_blk, (void*)&c->cell_base,
                     (void*)&c->cell_first, (void*)&c->cell_end, (void*)&c->cell_level, (void*)&c->cell_child,
                     (void*)&c->cell_info, (void*)&c->leaf_count, (void*)&c->cell_list, (void*)&cap, (void*)&c->g };
    FF_CUDA(c, cudaLaunchCooperativeKernel((const void*)ff_k_build, dim3(blocks), dim3(FF_BUILD_THREADS), args, 0,
                                           c->stream));
    c->launches++;
    return FF_OK;
}

int ff_launch_moments(ff_ctx* c, const float* mom)
{
    int n = (int)c->n;
    const int quad = c->order == 1 ? 1 : 0;
    const void* kernel = quad ? (const void*)ff_k_moments<true> : (const void*)ff_k_moments<false>;
    int& per_sm = c->occ_moments[quad];
    if (!per_sm) {
        if (quad) FF_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ff_k_moments<true>, FF_MOM_THREADS, 0));
        else FF_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ff_k_moments<false>, FF_MOM_THREADS, 0));
        if (per_sm < 1) return FF_ERR_CUDA;
    }
    int blocks = min((n + FF_MOM_THREADS - 1) / FF_MOM_THREADS, c->num_sms * min(per_sm, 8));
    const uint32_t* perm = c->idx[0];
    void* args[] = { (void*)&mom, (void*)&perm, (void*)&n, (void*)&c->g, (void*)&c->cell_first, (void*)&c->cell_end,
                     (void*)&c->cell_list, (void*)&c->cell_child, (void*)&c->leaf_count, (void*)&c->pos_s,
                     (void*)&c->mom_s, (void*)&c->cell_sums, (void*)&c->cell_centre,
                     (void*)&c->cell_moment, (void*)&c->cell_sums2, (void*)&c->cell_quad };
    FF_CUDA(c, cudaLaunchCooperativeKernel(kernel, dim3(blocks), dim3(FF_MOM_THREADS), args, 0, c->stream));
    c->launches++;
    return FF_OK;
}
